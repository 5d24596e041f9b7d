// dm_fast.cuh -- optimised forward mesh-FT kernels (rows A1-A4 of the hot path), sm_100a.
//
// Formulation.  With nodes x_0,x_1,x_2 = k.v_0, k.v_1, k.v_2 of a triangle, eq. 9
// reads  g = sum_j c_j e^{-i x_j},  c_j = -1 / prod_{m != j} (x_j - x_m)  -- REAL coefficients.  Summed over the mesh,
//     F(k) = sum_v e^{-i k.v} C_v(k),      C_v(k) = sum_{T containing v} s_T(k) c_{T,v}(k),
// so the complex exponential is needed once per (frequency, vertex visit), not once per (frequency, triangle corner).
// The mesh is walked as triangle strips (dm_strips.h): a vertex stays in a 3-slot register window while the (up to
// three) consecutive strip triangles that contain it add their real coefficients; when it leaves the window its phase
// is applied once:  F += e^{-ik.v} C_v.   Per (triangle, frequency) pair this costs ~18 FP32 instructions and one
// MUFU.RCP instead of three complex exponentials.
//
// Thread layout: one thread owns DM_K consecutive SIGNED y-frequencies of one (i_x, i_z); its phases advance along the
// run by one complex rotation rho_v = e^{-i kstep_y v_y} per step (exact start phase from integer turns, then <= DM_K-1
// rotations, so no long recurrences).  A warp = 32 consecutive i_z (coalesced stores); a CTA walks one chunk of strip
// records staged through shared memory.
//
// Numerical stability (reading R4).  eq. 9's cancellation error is ~ eps (|d1|+|d2|+|d3|)/|d1 d2 d3|
// (d = gaps, eps ~ 1e-6 the phase accuracy).  A pair whose gap product |d1 d2 d3| is below tau is EXCLUDED from the fast
// sum (its reciprocal is forced to zero) and flagged; after each tile every thread re-evaluates its flagged pairs
// through the robust series / far-pair branches of dm_math.cuh (compacted per lane, so the divergent work is only the
// flagged pairs).  Frequencies so low that EVERY triangle has small gaps (|k| h_max < DM_LOWK_RADIUS) skip the fast
// kernel and go to dm_k_forward_lowk, which evaluates all their pairs with the robust branches.
#pragma once
#include "dm_kernels.cuh"
#include "dm_strips.h"

static_assert(DM_STRIP_UNROLL == 6, "the strip loop is unrolled by 6 (window period 3 x gap ping-pong 2)");
#define DM_K 8                      // frequencies per thread (run along y)
#define DM_FAST_THREADS 128
#ifndef DM_FAST_MINCTA
#define DM_FAST_MINCTA 3            // resident CTAs per SM the register allocation aims at (160 registers: faster than 4 x 128)
#endif
#ifndef DM_FAST_TILE
#define DM_FAST_TILE 384            // strip records per shared-memory tile (multiple of DM_STRIP_UNROLL and of 32)
#endif
#define DM_FORCE_KH2 361.0f          // (|k| h_T)^2 above which a face skips the fast path of the forward kernel
#define DM_FORCE_OUTLIER_KH2 64.0f   // the same for a face whose longest edge is an outlier of the mesh:
#define DM_FORCE_OUTLIER_RATIO2 6.25f //   h_T^2 > 6.25 h_rms^2
#define DM_LOWK_RADIUS 0.5f         // |k| h_max below which a frequency is "low" (all gaps small for all triangles)
#define DM_LOWK_BOX 24              // low-k kernel covers |n_a| <= DM_LOWK_BOX
#ifndef DM_FAST_MIN_CHUNK
#define DM_FAST_MIN_CHUNK 16        // fewest faces per strip chunk (host policy of dm_plan_create)
#endif

// strip record = 3 x float4 (48 B):
//   r0 = (u_ret.xyz [uint32 bit patterns], rho_ret.re)     retiring vertex: fixed-point position, y-rotation
//   r1 = (rho_ret.im, e.xyz)                               e = v_new - v_prev
//   r2 = surface: (|m_T|, 0, 0, h2)   volume: (m_T.xyz, h2)  x..z zero when the step closes no triangle; h2 = longest
//        squared edge of the face
struct DmStripDev {
    const int32_t* vid_new;
    const int32_t* vid_prev;
    const int32_t* vid_ret;
    const int32_t* fid;
    int n_rec;
};

// ---- A1 for strips: records from the current vertex positions ----------------------------------------------------
__global__ void dm_k_strip_geometry(const float* __restrict__ vertices, const int32_t* __restrict__ faces, DmStripDev st,
                                    DmGridDev grid, int mode, float4* __restrict__ rec, unsigned int* __restrict__ hmax2_bits)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    float h2 = 0.f, e2sum = 0.f;
    if (i < st.n_rec) {
        const int vn = st.vid_new[i], vp = st.vid_prev[i], vr = max(st.vid_ret[i], 0), f = st.fid[i];
        uint32_t u[3];
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            double tt = (double)vertices[3 * vr + d] * grid.inv_len[d];
            tt -= floor(tt);
            u[d] = (uint32_t)(unsigned long long)(tt * 4294967296.0 + 0.5);
        }
        // rho = e^{-2 pi i v_y / L_y}: one step of n_y
        double ty = (double)vertices[3 * vr + 1] * grid.inv_len[1];
        ty -= rint(ty);
        double sn, cs;
        sincospi(2.0 * ty, &sn, &cs);
        float e[3] = {0.f, 0.f, 0.f};
        if (vp >= 0) {
#pragma unroll
            for (int d = 0; d < 3; ++d) e[d] = vertices[3 * vn + d] - vertices[3 * vp + d];
        }
        float4 r2 = make_float4(0.f, 0.f, 0.f, 0.f);
        if (f >= 0) {
            const int i1 = faces[3 * f], i2 = faces[3 * f + 1], i3 = faces[3 * f + 2];
            float a[3], b[3];
#pragma unroll
            for (int d = 0; d < 3; ++d) {
                a[d] = vertices[3 * i2 + d] - vertices[3 * i1 + d];
                b[d] = vertices[3 * i3 + d] - vertices[3 * i1 + d];
            }
            float m[3];
            dm_cross(a, b, m);
            const float wf = grid.face_w ? grid.face_w[f] : 1.0f;   // density weight of the face
            if (mode == 1) r2 = make_float4(wf * sqrtf(m[0] * m[0] + m[1] * m[1] + m[2] * m[2]), 0.f, 0.f, 0.f);
            else r2 = make_float4(wf * m[0], wf * m[1], wf * m[2], 0.f);
            // longest edge of the triangle (squared) and the sum of its squared edges
            const float c[3] = {b[0] - a[0], b[1] - a[1], b[2] - a[2]};
            const float a2 = a[0] * a[0] + a[1] * a[1] + a[2] * a[2], b2 = b[0] * b[0] + b[1] * b[1] + b[2] * b[2],
                        c2 = c[0] * c[0] + c[1] * c[1] + c[2] * c[2];
            h2 = fmaxf(fmaxf(a2, b2), c2);
            e2sum = a2 + b2 + c2;
            r2.w = h2;   // longest squared edge of the face: a face that is coarse for the grid skips the fast path
        }
        rec[3 * (size_t)i + 0] = make_float4(__uint_as_float(u[0]), __uint_as_float(u[1]), __uint_as_float(u[2]), (float)cs);
        rec[3 * (size_t)i + 1] = make_float4((float)(-sn), e[0], e[1], e[2]);
        rec[3 * (size_t)i + 2] = r2;
    }
    dm_edge_stats_add(hmax2_bits, h2, e2sum, grid.edge_fix);
}

// "low" frequencies: |k| h_max < DM_LOWK_RADIUS (every triangle has only small gaps there) and inside the box the
// low-k kernel covers.  Decided per frequency; the fast kernel skips them, dm_k_forward_lowk owns them.
__device__ __forceinline__ bool dm_k_is_low(const DmGridDev& grid, int nx, int nys, int nz, float hmax2)
{
    if (abs(nx) > DM_LOWK_BOX || abs(nys) > DM_LOWK_BOX || nz > DM_LOWK_BOX) return false;
    const float kx = grid.kstep[0] * nx, ky = grid.kstep[1] * nys, kz = grid.kstep[2] * nz;
    return (kx * kx + ky * ky + kz * kz) * hmax2 < DM_LOWK_RADIUS * DM_LOWK_RADIUS;
}

__device__ __forceinline__ float dm_rcp_ftz(float x)
{
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// The gap of a strip edge at one frequency of the run -- ONE definition, used by the fast loop and by the slow-path
// re-evaluation, so both take bit-identical decisions (explicit roundings: no contraction differences).
__device__ __forceinline__ float dm_edge_gxz(float kx, float kz, float ex, float ez) { return __fmaf_rn(kx, ex, __fmul_rn(kz, ez)); }
__device__ __forceinline__ float dm_edge_gap(float kyj, float ey, float gxz) { return __fmaf_rn(kyj, ey, gxz); }
__device__ __forceinline__ float dm_gap_product(float dp, float dn, float& df)
{
    df = __fadd_rn(dp, dn);
    return __fmul_rn(__fmul_rn(dp, dn), df);
}

// ---- A3/A4 forward, fast kernel ---------------------------------------------------------------------------------
// grid = (k-blocks of DM_FAST_THREADS threads, n_chunks).  part[chunk][k] receives this chunk's partial sum, already
// multiplied by the volume-mode prefactor i/|k|^2.
template <int MODE>
__global__ void __launch_bounds__(DM_FAST_THREADS, DM_FAST_MINCTA)
dm_k_forward_fast(const float4* __restrict__ rec, const int32_t* __restrict__ chunk_off, DmGridDev grid, int ix_begin,
                  int ix_end, int n_yruns, float tau, const unsigned int* __restrict__ hmax2_bits, size_t part_stride,
                  float2* __restrict__ part)
{
    __shared__ float4 tile[(DM_FAST_TILE + 1) * 3];              // +1: halo record (edge of the step before the tile)
    __shared__ uint32_t flagw[(DM_FAST_TILE / 32) * DM_FAST_THREADS];
    const int tid = threadIdx.x;
    // one thread per (i_x, y-run, i_z); under the narrow band only the listed threads (those with a frequency in the band)
    const long long n_thr = grid.band_slots ? (long long)grid.n_band_slots : (long long)(ix_end - ix_begin) * n_yruns * grid.nzh;
    const long long lin = (long long)blockIdx.x * DM_FAST_THREADS + tid;
    bool in_range = lin < n_thr;
    const long long l = in_range ? lin : 0;
    int iz, yrun, ix;
    if (grid.band_slots) {
        const uint32_t s = grid.band_slots[l];
        iz = (int)(s & 511u);
        yrun = (int)((s >> 9) & 2047u);
        ix = (int)(s >> 20);
        in_range = in_range && ix >= ix_begin && ix < ix_end;
    } else {
        iz = (int)(l % grid.nzh);
        yrun = (int)((l / grid.nzh) % n_yruns);
        ix = ix_begin + (int)(l / ((long long)grid.nzh * n_yruns));
    }
    const int nx = dm_signed_freq(ix, grid.nx), nz = iz;
    const int nys0 = -(grid.ny / 2) + yrun * DM_K;               // first signed y-frequency of the run
    const float hmax2 = __uint_as_float(*hmax2_bits), hmean2 = dm_edge_mean2(hmax2_bits, grid);
    const float kx = grid.kstep[0] * nx, kz = grid.kstep[2] * nz;
    float kyj[DM_K], tauj[DM_K];    // tauj < 0 switches a low frequency off (never flagged; its sums are not stored)
    // On a mesh that is coarse for the grid (|k| h >> 1) the rounding error of a gap k.e grows like |k| h while the
    // triangle integral itself decays like 1/(|k| h)^2, so the threshold scales with max(1, (|k| h_rms / 10)^3): exactly 1 on
    // meshes whose edges are a few voxels long (the benchmark configurations), larger on coarse meshes.
    // One value per thread, taken at the largest |k| of its run.
    const float kye = fmaxf(fabsf(grid.kstep[1] * (float)nys0), fabsf(grid.kstep[1] * (float)(nys0 + DM_K - 1)));
    const float k2t = kx * kx + kye * kye + kz * kz;          // largest |k|^2 of the thread's run
    const float kh2 = 0.01f * k2t * hmean2;                   // (|k| h_rms / 10)^2
    // A mesh whose longest edge is far above its RMS edge (stretched meshes, outlier faces) shrinks the ball the low-k
    // kernel owns (|k| h_max < DM_LOWK_RADIUS), so this kernel meets frequencies at which most faces have three small
    // gaps: the threshold grows with h_max / h_rms - 1.5, between 1 (h_max <= 2.5 h_rms: the benchmark meshes) and 16.
    const float ar = fminf(fmaxf(sqrtf(hmax2 / fmaxf(hmean2, 1e-30f)) - 1.5f, 1.0f), 16.0f);
    const float tau_t = tau * ar * fmaxf(1.0f, kh2 * sqrtf(kh2));
    // Longest squared edge above which a face skips the fast path at this thread's frequencies: |k| h_T > 19 for any
    // face, |k| h_T > 8 already for a face that is an outlier of its mesh (h_T > 2.5 h_rms: none on the benchmark meshes).
    // Such a face can have one gap of the order of its own rounding error while |pqr| is still far above tau.
    const float ik2t = 1.0f / fmaxf(k2t, 1e-30f);
    const float force_h2 = fminf(DM_FORCE_KH2 * ik2t, fmaxf(DM_FORCE_OUTLIER_KH2 * ik2t, DM_FORCE_OUTLIER_RATIO2 * hmean2));
    bool live = false;
#pragma unroll
    for (int j = 0; j < DM_K; ++j) {
        kyj[j] = __fmul_rn(grid.kstep[1], (float)(nys0 + j));
        const bool low = dm_k_is_low(grid, nx, nys0 + j, nz, hmax2) || !dm_in_band(grid, nx, nys0 + j, nz);
        tauj[j] = low ? -1.0f : tau_t;
        live |= !low;
    }
    live &= in_range;
    if (!__syncthreads_or(live ? 1 : 0)) return;   // nothing to do for this block of frequencies (narrow band)

    float Fre[DM_K], Fim[DM_K];     // running sums (tile sums of the fast path + slow-path pairs)
    float C0[DM_K], C1[DM_K], dp[DM_K];
#pragma unroll
    for (int j = 0; j < DM_K; ++j) Fre[j] = Fim[j] = C0[j] = C1[j] = dp[j] = 0.f;

    const int rec_begin = chunk_off[blockIdx.y], rec_end = chunk_off[blockIdx.y + 1];
    for (int t0 = rec_begin; t0 < rec_end; t0 += DM_FAST_TILE) {
        const int cnt = min(DM_FAST_TILE, rec_end - t0);        // multiple of DM_STRIP_UNROLL
        __syncthreads();
        // tile[0] = halo (record t0-1, or zeros at the chunk start), tile[1+s] = record t0+s
        for (int i = tid; i < (cnt + 1) * 3; i += DM_FAST_THREADS) {
            const long long src = 3LL * (t0 - 1) + i;
            tile[i] = (t0 == rec_begin && i < 3) ? make_float4(0.f, 0.f, 0.f, 0.f) : rec[src];
        }
        __syncthreads();
        if (live) {
            float Tre[DM_K], Tim[DM_K];  // per-tile sums keep the long accumulation accurate
#pragma unroll
            for (int j = 0; j < DM_K; ++j) Tre[j] = Tim[j] = 0.f;
            uint32_t word = 0;
#pragma unroll 6
            for (int s = 0; s < cnt; ++s) {
                const float4 r0 = tile[3 * (s + 1)], r1 = tile[3 * (s + 1) + 1], r2 = tile[3 * (s + 1) + 2];
                cf E = dm_expmi_turns_fast(dm_phase_turns(nx, nys0, nz, __float_as_uint(r0.x), __float_as_uint(r0.y),
                                                          __float_as_uint(r0.z)));
                const cf rho = {r0.w, r1.x};
                const float gxz = dm_edge_gxz(kx, kz, r1.y, r1.w);
                // a face that is coarse for this frequency (h_T^2 > force_h2 above) contributes
                // nothing here and goes to the robust branches whole
                const bool force = r2.w > force_h2;
                const float r2x = force ? 0.f : r2.x, r2y = force ? 0.f : r2.y;
                float mxz = 0.f;
                if (MODE == 0) mxz = force ? 0.f : fmaf(kx, r2.x, kz * r2.z);
                bool any_bad = force;
#pragma unroll
                for (int j = 0; j < DM_K; ++j) {
                    const float dn = dm_edge_gap(kyj[j], r1.z, gxz);
                    float df;
                    const float pr = dm_gap_product(dp[j], dn, df);
                    const bool bad = !(fabsf(pr) > tauj[j]);   // also catches pr = 0 when tau = 0 (0 * rcp(0) would be NaN)
                    any_bad |= bad;
                    float sc = (MODE == 1) ? r2x : fmaf(kyj[j], r2y, mxz);
                    sc = bad ? 0.f : sc * dm_rcp_ftz(pr);
                    // nodes x0 = v_ret, x1 = v_prev, x2 = v_new; gaps p = dp, r = dn, q = df:
                    //   c0 = -r/(pqr), c1 = +q/(pqr), c2 = -p/(pqr)
                    const float c0 = fmaf(-dn, sc, C0[j]);
                    C0[j] = fmaf(df, sc, C1[j]);
                    C1[j] = -dp[j] * sc;
                    dp[j] = dn;
                    Tre[j] = fmaf(E.re, c0, Tre[j]);
                    Tim[j] = fmaf(E.im, c0, Tim[j]);
                    E = cmul(E, rho);
                }
                word |= (any_bad ? 1u : 0u) << (s & 31);
                if ((s & 31) == 31) {
                    flagw[(s >> 5) * DM_FAST_THREADS + tid] = word;
                    word = 0;
                }
            }
            if ((cnt & 31) != 0) flagw[(cnt >> 5) * DM_FAST_THREADS + tid] = word;
#pragma unroll
            for (int j = 0; j < DM_K; ++j) {
                Fre[j] += Tre[j];
                Fim[j] += Tim[j];
            }
            // ---- slow path: re-evaluate this thread's flagged pairs of the tile through the robust branches ----------
            const int n_words = (cnt + 31) >> 5;
            for (int w = 0; w < n_words; ++w) {
                uint32_t bits = flagw[w * DM_FAST_THREADS + tid];
                while (bits) {
                    const int s = (w << 5) + __ffs(bits) - 1;
                    bits &= bits - 1;
                    const float4 r2 = tile[3 * (s + 1) + 2];
                    const bool valid = (MODE == 1) ? (r2.x != 0.f) : (r2.x != 0.f || r2.y != 0.f || r2.z != 0.f);
                    if (!valid) continue;
                    const float4 r0 = tile[3 * (s + 1)], r1 = tile[3 * (s + 1) + 1], q1 = tile[3 * s + 1];
                    const float gn = dm_edge_gxz(kx, kz, r1.y, r1.w), gp = dm_edge_gxz(kx, kz, q1.y, q1.w);
                    const bool force = r2.w > force_h2;   // the whole record was left to this path
                    uint32_t mask = 0;
#pragma unroll
                    for (int j = 0; j < DM_K; ++j) {
                        float df;
                        const float pr = dm_gap_product(dm_edge_gap(kyj[j], q1.z, gp), dm_edge_gap(kyj[j], r1.z, gn), df);
                        mask |= (((force && tauj[j] >= 0.f) || !(fabsf(pr) > tauj[j])) ? 1u : 0u) << j;
                    }
                    while (mask) {
                        const int j = __ffs(mask) - 1;
                        mask &= mask - 1;
                        const float ky = __fmul_rn(grid.kstep[1], (float)(nys0 + j));
                        const float p = dm_edge_gap(ky, q1.z, gp);            // x1 - x0
                        const float q = __fadd_rn(p, dm_edge_gap(ky, r1.z, gn));  // x2 - x0
                        const cf psi = dm_psi_value_fast(p, q);
                        const cf E = dm_expmi_turns_fast(dm_phase_turns(nx, nys0 + j, nz, __float_as_uint(r0.x),
                                                                        __float_as_uint(r0.y), __float_as_uint(r0.z)));
                        const float sc = (MODE == 1) ? r2.x : fmaf(kx, r2.x, fmaf(ky, r2.y, kz * r2.z));
                        const cf g = cscale(cmul(E, psi), sc);
#pragma unroll
                        for (int jj = 0; jj < DM_K; ++jj)
                            if (jj == j) {
                                Fre[jj] += g.re;
                                Fim[jj] += g.im;
                            }
                    }
                }
            }
        }
    }
    if (live) {
        float2* out = part + (size_t)blockIdx.y * part_stride;
#pragma unroll
        for (int j = 0; j < DM_K; ++j) {
            const int nys = nys0 + j;
            if (nys > (grid.ny - 1) / 2 || tauj[j] < 0.f) continue;  // ragged last run / owned by the low-k kernel
            const int iy = nys < 0 ? nys + grid.ny : nys;
            float re = Fre[j], im = Fim[j];
            if (MODE == 0) {
                const float k2 = kx * kx + kyj[j] * kyj[j] + kz * kz;
                const float ik2 = (k2 > 0.f) ? 1.0f / k2 : 0.f;
                const float t = re;
                re = -im * ik2;
                im = t * ik2;
            }
            out[((size_t)ix * grid.ny + iy) * grid.nzh + iz] = make_float2(re, im);
        }
    }
}

// ---- A4 at low |k|: every pair through the robust branches; one CTA per low frequency, threads stride over the records ----
// Candidates are the (2 bx + 1)(2 by + 1)(bz + 1) frequencies |n_x| <= bx, |n_y| <= by, n_z <= bz (the low-k box clipped to the
// grid).  Every THREAD of the grid tests one candidate (interleaved over the CTAs, so that the low ball around k = 0 is spread
// over all of them); a CTA then evaluates the low ones it found, one after the other, with all its threads.  Each frequency
// is written by exactly one CTA and its block sum is taken in a fixed order (lane tree, then the warps in order), so the
// result does not depend on the order in which a CTA lists its frequencies.  grid = ceil(candidates / DM_LOWK_CAND).
#define DM_LOWK_THREADS 256
#define DM_LOWK_CAND 64            // candidates tested per CTA (by its first threads): enough CTAs to balance the low ones
template <int MODE>
__global__ void __launch_bounds__(DM_LOWK_THREADS)
dm_k_forward_lowk(const float4* __restrict__ rec, const int32_t* __restrict__ chunk_off, int n_chunks, DmGridDev grid,
                  int ix_begin, int ix_end, int bx, int by, int bz, const unsigned int* __restrict__ hmax2_bits,
                  float2* __restrict__ F)
{
    __shared__ float wsum[2][DM_LOWK_THREADS / 32];
    __shared__ int list[DM_LOWK_CAND];
    __shared__ int n_list;
    const int lane = threadIdx.x & 31, wrp = threadIdx.x >> 5;
    const int Wy = 2 * by + 1, n_cand = (2 * bx + 1) * Wy * (bz + 1);
    const float hmax2 = __uint_as_float(*hmax2_bits);
    if (threadIdx.x == 0) n_list = 0;
    __syncthreads();
    {
        const int fi = (int)threadIdx.x * (int)gridDim.x + (int)blockIdx.x;
        if (threadIdx.x < DM_LOWK_CAND && fi < n_cand) {
            const int nz = fi % (bz + 1), nys = (fi / (bz + 1)) % Wy - by, nx = fi / ((bz + 1) * Wy) - bx;
            const int ix = nx < 0 ? nx + grid.nx : nx;
            const bool on_grid = !(nz > grid.nz / 2 || nys < -(grid.ny / 2) || nys > (grid.ny - 1) / 2 || nx < -(grid.nx / 2) ||
                                   nx > (grid.nx - 1) / 2) && ix >= ix_begin && ix < ix_end;
            if (on_grid && dm_k_is_low(grid, nx, nys, nz, hmax2) && dm_in_band(grid, nx, nys, nz)) list[atomicAdd(&n_list, 1)] = fi;
        }
    }
    __syncthreads();
    const int n_mine = n_list;
    for (int li = 0; li < n_mine; ++li) {
        const int fi = list[li];
        const int nz = fi % (bz + 1), nys = (fi / (bz + 1)) % Wy - by, nx = fi / ((bz + 1) * Wy) - bx;
        const int ix = nx < 0 ? nx + grid.nx : nx, iy = nys < 0 ? nys + grid.ny : nys;
        const float kx = grid.kstep[0] * nx, ky = grid.kstep[1] * nys, kz = grid.kstep[2] * nz;
        float are = 0.f, aim = 0.f;
        for (int c = 0; c < n_chunks; ++c) {
            const int b = chunk_off[c], e = chunk_off[c + 1];
            for (int i = b + 1 + (int)threadIdx.x; i < e; i += DM_LOWK_THREADS) {   // record b closes no triangle
                const float4 r2 = rec[3 * (size_t)i + 2];
                const bool valid = (MODE == 1) ? (r2.x != 0.f) : (r2.x != 0.f || r2.y != 0.f || r2.z != 0.f);
                if (!valid) continue;
                const float4 r0 = rec[3 * (size_t)i], r1 = rec[3 * (size_t)i + 1], q1 = rec[3 * (size_t)i - 2];
                const float p = fmaf(kx, q1.y, fmaf(ky, q1.z, kz * q1.w));
                const float q = p + fmaf(kx, r1.y, fmaf(ky, r1.z, kz * r1.w));
                cf psi, d1, d2;
                dm_psi_robust<false>(p, q, psi, d1, d2);
                const cf E = dm_expmi_turns(dm_phase_turns(nx, nys, nz, __float_as_uint(r0.x), __float_as_uint(r0.y),
                                                           __float_as_uint(r0.z)));
                const float sc = (MODE == 1) ? r2.x : fmaf(kx, r2.x, fmaf(ky, r2.y, kz * r2.z));
                const cf g = cmul(E, psi);
                are = fmaf(sc, g.re, are);
                aim = fmaf(sc, g.im, aim);
            }
        }
        for (int o = 16; o > 0; o >>= 1) {
            are += __shfl_xor_sync(0xffffffffu, are, o);
            aim += __shfl_xor_sync(0xffffffffu, aim, o);
        }
        __syncthreads();   // the previous frequency's sums have been read
        if (lane == 0) {
            wsum[0][wrp] = are;
            wsum[1][wrp] = aim;
        }
        __syncthreads();
        if (threadIdx.x == 0) {
            are = 0.f, aim = 0.f;
#pragma unroll
            for (int w = 0; w < DM_LOWK_THREADS / 32; ++w) {
                are += wsum[0][w];
                aim += wsum[1][w];
            }
            if (MODE == 0) {
                const float k2 = kx * kx + ky * ky + kz * kz;
                const float ik2 = (k2 > 0.f) ? 1.0f / k2 : 0.f;
                const float t = are;
                are = -aim * ik2;
                aim = t * ik2;
            }
            F[((size_t)ix * grid.ny + iy) * grid.nzh + nz] = make_float2(are, aim);
        }
    }
}

// ---- sum the chunk partials (fixed order) into F for every frequency the fast kernel owns ---------------------------
__global__ void dm_k_forward_finish(const float2* __restrict__ part, size_t part_stride, int n_chunks, DmGridDev grid,
                                    int ix_begin, int ix_end, const unsigned int* __restrict__ hmax2_bits,
                                    float2* __restrict__ F)
{
    const long long n_slab = (long long)(ix_end - ix_begin) * grid.ny * grid.nzh;
    const long long l = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (l >= n_slab) return;
    const int iz = (int)(l % grid.nzh), iy = (int)((l / grid.nzh) % grid.ny);
    const int ix = ix_begin + (int)(l / ((long long)grid.nzh * grid.ny));
    const int nx = dm_signed_freq(ix, grid.nx), nys = dm_signed_freq(iy, grid.ny);
    const size_t o = ((size_t)ix * grid.ny + iy) * grid.nzh + iz;
    if (!dm_in_band(grid, nx, nys, iz)) {   // narrow band: skipped entries are zero
        F[o] = make_float2(0.f, 0.f);
        return;
    }
    if (dm_k_is_low(grid, nx, nys, iz, __uint_as_float(*hmax2_bits))) return;
    float re = 0.f, im = 0.f;
    for (int c = 0; c < n_chunks; ++c) {
        const float2 v = part[(size_t)c * part_stride + o];
        re += v.x;
        im += v.y;
    }
    F[o] = make_float2(re, im);
}
