// dm_kernels.cuh -- CUDA kernels of the mesh Fourier transform (sm_100a), reference-quality "robust" variants.
//
// These kernels evaluate EVERY (triangle, frequency) pair through the robust branches of dm_math.cuh.  They are the
// always-correct path and the slow path of the optimised kernels; see DESIGN.md section 5 for the kernel list.
//
// Notation: triangle T = (v1,v2,v3), eb = v2-v1, ec = v3-v1, m_T = eb x ec = 2 A_T N_T,
// a = k.v1, p = k.eb, q = k.ec, g = e^{-ia} psi(p,q).  Stored frequency (ix,iy,iz) -> integers (nx,ny,nz), k_a = kstep_a n_a.
#pragma once
#include "dm_math.cuh"

// One triangle record = 4 x float4 (64 B), rebuilt every call because vertices move (row A1).
//   r0 = (ux, uy, uz [uint32 bit patterns: v1/L in fixed-point turns], |m_T|)
//   r1 = (eb.xyz, 0)   r2 = (ec.xyz, 0)   r3 = (m_T.xyz, 0)
struct DmGridDev {
    int nx, ny, nz, nzh;      // voxels and nz/2+1
    float kstep[3];           // 2 pi / L_a
    double inv_len[3];        // 1 / L_a
    // narrow band: only frequencies with 1/2 k^T B k < band_lim are evaluated (h_hat(k) > cutoff for
    // the Gaussian PSF of covariance B, band_lim = ln(1/cutoff)); band_lim = +inf switches the band off
    float band_cov[6];        // xx yy zz xy xz yz
    float band_lim;
    float edge_fix;           // fixed-point scale of the squared edge lengths summed by the geometry kernels
    float inv_edge_norm;      // 1 / (3 n_faces edge_fix): mean squared edge = sum * inv_edge_norm
    const float* face_w;      // per-face density weights, device [n_faces]; nullptr = all 1
    const uint32_t* band_slots;  // narrow band: the forward kernel's active threads, packed i_x << 20 | y-run << 9 | i_z
    int n_band_slots;            // (device, built by dm_plan_set_narrow_band); nullptr / 0 without a band
    int nzb;                  // stored z-frequencies 0..nzb-1 can be inside the band (nzb = nzh when the band is off)
};

// Edge statistics of the mesh, rebuilt by the geometry kernel of every call in a 16-byte device buffer:
//   word 0 = longest squared edge (float bits; non-negative floats order like their bit patterns), bytes 8..15 = sum of
//   the squared edges of all faces in fixed point (integer adds: the sum does not depend on the order of the atomics).
// dm_edge_stats_add is called by every thread of a warp (val = 0, h2 = 0 for threads without a face).
__device__ __forceinline__ void dm_edge_stats_add(unsigned int* stats, float h2max, float e2sum, float edge_fix)
{
    unsigned long long s = (unsigned long long)(e2sum * edge_fix);
    for (int o = 16; o > 0; o >>= 1) {
        h2max = fmaxf(h2max, __shfl_xor_sync(0xffffffffu, h2max, o));
        s += __shfl_xor_sync(0xffffffffu, s, o);
    }
    if ((threadIdx.x & 31) == 0 && h2max > 0.f) {
        atomicMax(stats, __float_as_uint(h2max));
        atomicAdd(reinterpret_cast<unsigned long long*>(stats) + 1, s);
    }
}
// mean squared edge length of the mesh
__device__ __forceinline__ float dm_edge_mean2(const unsigned int* stats, const DmGridDev& grid)
{
    return (float)(reinterpret_cast<const unsigned long long*>(stats)[1]) * grid.inv_edge_norm;
}

__device__ __forceinline__ bool dm_in_band(const DmGridDev& grid, int nx, int ny, int nz)
{
    const float kx = grid.kstep[0] * nx, ky = grid.kstep[1] * ny, kz = grid.kstep[2] * nz;
    const float quad = grid.band_cov[0] * kx * kx + grid.band_cov[1] * ky * ky + grid.band_cov[2] * kz * kz +
                       2.0f * (grid.band_cov[3] * kx * ky + grid.band_cov[4] * kx * kz + grid.band_cov[5] * ky * kz);
    return nz < grid.nzb && 0.5f * quad < grid.band_lim;
}

__device__ __forceinline__ int dm_signed_freq(int i, int n) { return (i < (n + 1) / 2) ? i : i - n; }

// ---- A1: per-triangle geometry pre-pass --------------------------------------------------------------------------
__global__ void dm_k_geometry(const float* __restrict__ vertices, const int32_t* __restrict__ faces, int n_faces,
                              DmGridDev grid, float4* __restrict__ rec)
{
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= n_faces) return;
    const int i1 = faces[3 * t], i2 = faces[3 * t + 1], i3 = faces[3 * t + 2];
    const float v1[3] = {vertices[3 * i1], vertices[3 * i1 + 1], vertices[3 * i1 + 2]};
    const float v2[3] = {vertices[3 * i2], vertices[3 * i2 + 1], vertices[3 * i2 + 2]};
    const float v3[3] = {vertices[3 * i3], vertices[3 * i3 + 1], vertices[3 * i3 + 2]};
    uint32_t u[3];
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        double tt = (double)v1[d] * grid.inv_len[d];
        tt -= floor(tt);
        u[d] = (uint32_t)(unsigned long long)(tt * 4294967296.0 + 0.5);  // wraps 2^32 -> 0
    }
    const float eb[3] = {v2[0] - v1[0], v2[1] - v1[1], v2[2] - v1[2]};
    const float ec[3] = {v3[0] - v1[0], v3[1] - v1[1], v3[2] - v1[2]};
    float m[3];
    dm_cross(eb, ec, m);
    const float wf = grid.face_w ? grid.face_w[t] : 1.0f;   // density weight of the face: scales m_T and |m_T|
    const float mn = wf * sqrtf(m[0] * m[0] + m[1] * m[1] + m[2] * m[2]);
    m[0] *= wf, m[1] *= wf, m[2] *= wf;
    rec[4 * (size_t)t + 0] = make_float4(__uint_as_float(u[0]), __uint_as_float(u[1]), __uint_as_float(u[2]), mn);
    rec[4 * (size_t)t + 1] = make_float4(eb[0], eb[1], eb[2], 0.f);
    rec[4 * (size_t)t + 2] = make_float4(ec[0], ec[1], ec[2], 0.f);
    rec[4 * (size_t)t + 3] = make_float4(m[0], m[1], m[2], 0.f);
}

// ---- A5: the k = 0 entry in fp64: volume 1/6 sum v1.(v2 x v3), or total area sum |m_T|/2 -------------------------
// Two stages, both with fixed-order tree reductions (deterministic): DM_DC_BLOCKS block sums, then one final block.
#define DM_DC_BLOCKS 64
__global__ void __launch_bounds__(256)
dm_k_dc_partial(const float* __restrict__ vertices, const int32_t* __restrict__ faces, int n_faces, int mode,
                const float* __restrict__ face_w, double* __restrict__ partial)
{
    __shared__ double sh[256];
    double acc = 0.0;
    for (int t = blockIdx.x * blockDim.x + threadIdx.x; t < n_faces; t += gridDim.x * blockDim.x) {
        const int i1 = faces[3 * t], i2 = faces[3 * t + 1], i3 = faces[3 * t + 2];
        const double a[3] = {vertices[3 * i1], vertices[3 * i1 + 1], vertices[3 * i1 + 2]};
        const double b[3] = {vertices[3 * i2], vertices[3 * i2 + 1], vertices[3 * i2 + 2]};
        const double c[3] = {vertices[3 * i3], vertices[3 * i3 + 1], vertices[3 * i3 + 2]};
        const double wf = face_w ? (double)face_w[t] : 1.0;
        if (mode == 0) {
            acc += wf * (a[0] * (b[1] * c[2] - b[2] * c[1]) + a[1] * (b[2] * c[0] - b[0] * c[2]) +
                    a[2] * (b[0] * c[1] - b[1] * c[0])) * (1.0 / 6.0);
        } else {
            const double e[3] = {b[0] - a[0], b[1] - a[1], b[2] - a[2]}, f[3] = {c[0] - a[0], c[1] - a[1], c[2] - a[2]};
            const double m[3] = {e[1] * f[2] - e[2] * f[1], e[2] * f[0] - e[0] * f[2], e[0] * f[1] - e[1] * f[0]};
            acc += wf * 0.5 * sqrt(m[0] * m[0] + m[1] * m[1] + m[2] * m[2]);
        }
    }
    sh[threadIdx.x] = acc;
    __syncthreads();
    for (int s = blockDim.x / 2; s > 0; s >>= 1) {
        if (threadIdx.x < s) sh[threadIdx.x] += sh[threadIdx.x + s];
        __syncthreads();
    }
    if (threadIdx.x == 0) partial[blockIdx.x] = sh[0];
}
__global__ void __launch_bounds__(DM_DC_BLOCKS)
dm_k_dc_final(const double* __restrict__ partial, float* __restrict__ F0, double* __restrict__ total)
{
    __shared__ double sh[DM_DC_BLOCKS];
    sh[threadIdx.x] = partial[threadIdx.x];
    __syncthreads();
    for (int s = DM_DC_BLOCKS / 2; s > 0; s >>= 1) {
        if (threadIdx.x < s) sh[threadIdx.x] += sh[threadIdx.x + s];
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        F0[0] = (float)sh[0];
        F0[1] = 0.f;
        *total = sh[0];   // volume or total area |Lambda| in fp64, kept for the area-normalised density (eq. 12)
    }
}

// ---- A3/A4 forward, robust variant: one thread per stored frequency, loop over all triangles ---------------------
#define DM_FWD_TILE 128
__global__ void __launch_bounds__(128)
dm_k_forward_robust(const float4* __restrict__ rec, int n_faces, DmGridDev grid, int mode, int ix_begin, int ix_end,
                    float2* __restrict__ F)
{
    __shared__ float4 tile[DM_FWD_TILE * 4];
    const long long n_slab = (long long)(ix_end - ix_begin) * grid.ny * grid.nzh;
    const long long lin = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const bool live = lin < n_slab;
    const long long l = live ? lin : 0;
    const int iz = (int)(l % grid.nzh);
    const int iy = (int)((l / grid.nzh) % grid.ny);
    const int ix = ix_begin + (int)(l / ((long long)grid.nzh * grid.ny));
    const int nx = dm_signed_freq(ix, grid.nx), ny = dm_signed_freq(iy, grid.ny), nz = iz;
    const float kx = grid.kstep[0] * nx, ky = grid.kstep[1] * ny, kz = grid.kstep[2] * nz;
    const float k2 = kx * kx + ky * ky + kz * kz;
    const float inv_k2 = (k2 > 0.f) ? 1.0f / k2 : 0.f;
    float acc_re = 0.f, acc_im = 0.f;
    for (int t0 = 0; t0 < n_faces; t0 += DM_FWD_TILE) {
        const int cnt = min(DM_FWD_TILE, n_faces - t0);
        __syncthreads();
        for (int i = threadIdx.x; i < cnt * 4; i += blockDim.x) tile[i] = rec[4 * (size_t)t0 + i];
        __syncthreads();
        float tre = 0.f, tim = 0.f;  // per-tile partial sums keep the long accumulation accurate
        for (int j = 0; j < cnt; ++j) {
            const float4 r0 = tile[4 * j], r1 = tile[4 * j + 1], r2 = tile[4 * j + 2];
            const float p = fmaf(kx, r1.x, fmaf(ky, r1.y, kz * r1.z));
            const float q = fmaf(kx, r2.x, fmaf(ky, r2.y, kz * r2.z));
            cf psi, d1, d2;
            dm_psi_robust<false>(p, q, psi, d1, d2);
            const cf E = dm_expmi_turns(dm_phase_turns(nx, ny, nz, __float_as_uint(r0.x), __float_as_uint(r0.y),
                                                       __float_as_uint(r0.z)));
            float w;
            if (mode == 1) {
                w = r0.w;
            } else {
                const float4 r3 = tile[4 * j + 3];
                w = fmaf(kx, r3.x, fmaf(ky, r3.y, kz * r3.z)) * inv_k2;
            }
            const cf g = cmul(E, psi);
            tre = fmaf(w, g.re, tre);
            tim = fmaf(w, g.im, tim);
        }
        acc_re += tre;
        acc_im += tim;
    }
    if (live) {
        const size_t o = ((size_t)ix * grid.ny + iy) * grid.nzh + iz;
        // volume mode carries the factor i of (i/|k|^2); entries outside the narrow band are zero
        if (!dm_in_band(grid, nx, ny, nz)) acc_re = acc_im = 0.f;
        F[o] = (mode == 1) ? make_float2(acc_re, acc_im) : make_float2(-acc_im, acc_re);
    }
}

// ---- A6 backward, robust variant: one thread per triangle, loop over a split of the stored frequencies ------------
// Per triangle and split it accumulates 13 real sums over k (kappa = conj(G) [surface] or i conj(G)/|k|^2 [volume],
// omega = 1 [surface] or k.m_T [volume]; g_b = dg/db, g_c = dg/dc; dg/da follows from  sum_p dg/da_p = -i g):
//   [0]      S0 = sum Re(kappa g)                    (surface: multiplies -w_p)
//   [1..3]   Q  = sum k Re(kappa g)                  (volume:  crossed with e_p)
//   [4..6]   W  = sum omega k Im(kappa g)            (= sum omega k Re(kappa (-i g)))
//   [7..9]   Vb = sum omega k Re(kappa g_b)
//   [10..12] Vc = sum omega k Re(kappa g_c)
// Layout of the partial sums: part[(split*13 + s)*n_faces + t].
#define DM_BWD_NSUM 13
__global__ void __launch_bounds__(128)
dm_k_backward_robust(const float4* __restrict__ rec, int n_faces, DmGridDev grid, int mode, int ix_begin, int ix_end,
                     int rows_per_split, const float2* __restrict__ G, float* __restrict__ part)
{
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    const bool live = t < n_faces;
    const int tt = live ? t : 0;
    const float4 r0 = rec[4 * (size_t)tt], r1 = rec[4 * (size_t)tt + 1], r2 = rec[4 * (size_t)tt + 2],
                 r3 = rec[4 * (size_t)tt + 3];
    const uint32_t ux = __float_as_uint(r0.x), uy = __float_as_uint(r0.y), uz = __float_as_uint(r0.z);
    const int n_rows = (ix_end - ix_begin) * grid.ny;
    const int row_begin = blockIdx.y * rows_per_split;
    const int row_end = min(n_rows, row_begin + rows_per_split);
    float acc[DM_BWD_NSUM];
#pragma unroll
    for (int s = 0; s < DM_BWD_NSUM; ++s) acc[s] = 0.f;
    for (int row = row_begin; row < row_end; ++row) {
        const int ix = ix_begin + row / grid.ny, iy = row % grid.ny;
        const int nx = dm_signed_freq(ix, grid.nx), ny = dm_signed_freq(iy, grid.ny);
        const float kx = grid.kstep[0] * nx, ky = grid.kstep[1] * ny;
        const float2* Grow = G + ((size_t)ix * grid.ny + iy) * grid.nzh;
        float racc[DM_BWD_NSUM];  // per-row partial sums
#pragma unroll
        for (int s = 0; s < DM_BWD_NSUM; ++s) racc[s] = 0.f;
        for (int iz = 0; iz < grid.nzh; ++iz) {
            const float kz = grid.kstep[2] * iz;
            float2 Gk = Grow[iz];
            if (!dm_in_band(grid, nx, ny, iz)) Gk = make_float2(0.f, 0.f);   // narrow band
            const float k2 = kx * kx + ky * ky + kz * kz;
            cf kappa;
            float omega;
            if (mode == 1) {
                kappa = {Gk.x, -Gk.y};
                omega = 1.0f;
            } else {
                const float inv_k2 = (k2 > 0.f) ? 1.0f / k2 : 0.f;
                kappa = {Gk.y * inv_k2, Gk.x * inv_k2};  // i conj(G) / |k|^2
                omega = fmaf(kx, r3.x, fmaf(ky, r3.y, kz * r3.z));
            }
            const float p = fmaf(kx, r1.x, fmaf(ky, r1.y, kz * r1.z));
            const float q = fmaf(kx, r2.x, fmaf(ky, r2.y, kz * r2.z));
            cf psi, dp, dq;
            dm_psi_robust<true>(p, q, psi, dp, dq);
            const cf E = dm_expmi_turns(dm_phase_turns(nx, ny, iz, ux, uy, uz));
            const cf kE = cmul(kappa, E);
            const cf kg = cmul(kE, psi);
            const float gb = kE.re * dp.re - kE.im * dp.im;  // Re(kappa g_b)
            const float gc = kE.re * dq.re - kE.im * dq.im;
            racc[0] += kg.re;
            racc[1] = fmaf(kx, kg.re, racc[1]);
            racc[2] = fmaf(ky, kg.re, racc[2]);
            racc[3] = fmaf(kz, kg.re, racc[3]);
            const float wi = omega * kg.im, wb = omega * gb, wc = omega * gc;
            racc[4] = fmaf(kx, wi, racc[4]);
            racc[5] = fmaf(ky, wi, racc[5]);
            racc[6] = fmaf(kz, wi, racc[6]);
            racc[7] = fmaf(kx, wb, racc[7]);
            racc[8] = fmaf(ky, wb, racc[8]);
            racc[9] = fmaf(kz, wb, racc[9]);
            racc[10] = fmaf(kx, wc, racc[10]);
            racc[11] = fmaf(ky, wc, racc[11]);
            racc[12] = fmaf(kz, wc, racc[12]);
        }
#pragma unroll
        for (int s = 0; s < DM_BWD_NSUM; ++s) acc[s] += racc[s];
    }
    if (live) {
#pragma unroll
        for (int s = 0; s < DM_BWD_NSUM; ++s) part[((size_t)blockIdx.y * DM_BWD_NSUM + s) * n_faces + t] = acc[s];
    }
}

// ---- A6 (end): sum the k-splits of every (sum, triangle) in fixed order into split 0's slot ---------------------------
// grid = (ceil(n_faces/128), 13): coalesced over triangles; a small mesh has hundreds of splits, which one thread per
// triangle would walk alone.
__global__ void __launch_bounds__(128)
dm_k_sum_splits(float* __restrict__ part, int n_faces, int n_split)
{
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= n_faces) return;
    const size_t o = (size_t)blockIdx.y * n_faces + t;
    float s = 0.f;
    for (int sp = 0; sp < n_split; ++sp) s += part[(size_t)sp * DM_BWD_NSUM * n_faces + o];
    part[o] = s;
}

// ---- A6 (end): sum the splits in fixed order and form the per-corner gradients ------------------------------------
//   surface (eq. 10):  grad_p = -w_p S0 + |m_T| V_p,     w_p = e_p x N_T, e_p = v_{p-} - v_{p+}
//   volume  (product rule, d(k.m_T)/dv_p = k x e_p):  grad_p = Q x e_p + V_p,  plus the k = 0 row
//            Re(G(0)) (v_{p+} x v_{p-})/6 when the slab holds it.
//   V_a = W - V_b - V_c.   Degenerate triangle in surface mode contributes 0 (reading R19).
__global__ void dm_k_corner_grads(const float* __restrict__ vertices, const int32_t* __restrict__ faces, int n_faces,
                                  int mode, int n_split, const float* __restrict__ part,
                                  const float2* __restrict__ G, int has_dc, const double* __restrict__ area_total,
                                  const double* __restrict__ sdot, int sdot_of_u, const float* __restrict__ face_w,
                                  float* __restrict__ corner)
{
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= n_faces) return;
    float s[DM_BWD_NSUM];
#pragma unroll
    for (int j = 0; j < DM_BWD_NSUM; ++j) s[j] = 0.f;
    for (int sp = 0; sp < n_split; ++sp)
#pragma unroll
        for (int j = 0; j < DM_BWD_NSUM; ++j) s[j] += part[((size_t)sp * DM_BWD_NSUM + j) * n_faces + t];
    if (area_total != nullptr) {
        // area-normalised density u = F/|Lambda| (eq. 12-13): the sums were taken with the cotangent G of
        // u, so  dL/dv = (1/|Lambda|) bare - (S/|Lambda|) d|Lambda|/dv,  S = sum_k Re(conj(G) u) = sdot/|Lambda|, and
        // d|Lambda|/dv_p = -w_p/2 folds into the coefficient of -w_p:  S0 -> S0/|Lambda| - S/(2|Lambda|)
        const double inv = 1.0 / *area_total;
#pragma unroll
        for (int j = 0; j < DM_BWD_NSUM; ++j) s[j] = (float)((double)s[j] * inv);
        // (*sdot = sum_k Re(conj(G) F) with the raw F, or with u = F/|Lambda| itself when sdot_of_u is set)
        s[0] = (float)((double)s[0] - 0.5 * (*sdot) * (sdot_of_u ? inv : inv * inv));
    }
    const int idx[3] = {faces[3 * t], faces[3 * t + 1], faces[3 * t + 2]};
    float v[3][3];
#pragma unroll
    for (int p = 0; p < 3; ++p)
#pragma unroll
        for (int d = 0; d < 3; ++d) v[p][d] = vertices[3 * idx[p] + d];
    float e[3][3];  // e_p = v_{p-} - v_{p+}
#pragma unroll
    for (int p = 0; p < 3; ++p)
#pragma unroll
        for (int d = 0; d < 3; ++d) e[p][d] = v[(p + 2) % 3][d] - v[(p + 1) % 3][d];
    const float ecv[3] = {-e[1][0], -e[1][1], -e[1][2]};   // v_3 - v_1
    float m[3];
    dm_cross(e[2], ecv, m);                                // (v_2 - v_1) x (v_3 - v_1) = m_T, as in the geometry pre-pass
    const float mn = sqrtf(m[0] * m[0] + m[1] * m[1] + m[2] * m[2]);
    float V[3][3];
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        V[1][d] = s[7 + d];
        V[2][d] = s[10 + d];
        V[0][d] = s[4 + d] - s[7 + d] - s[10 + d];
    }
    const float wf = face_w ? face_w[t] : 1.0f;   // density weight of the face
    float grad[3][3];
    if (mode == 1) {
        const float inv = (mn >= 1e-30f) ? 1.0f / mn : 0.f;
        const float N[3] = {m[0] * inv, m[1] * inv, m[2] * inv};
#pragma unroll
        for (int p = 0; p < 3; ++p) {
            const float w[3] = {e[p][1] * N[2] - e[p][2] * N[1], e[p][2] * N[0] - e[p][0] * N[2],
                                e[p][0] * N[1] - e[p][1] * N[0]};
#pragma unroll
            for (int d = 0; d < 3; ++d) grad[p][d] = (mn >= 1e-30f) ? wf * fmaf(mn, V[p][d], -w[d] * s[0]) : 0.f;
        }
    } else {
        const float Q[3] = {s[1], s[2], s[3]};
        const float g0 = has_dc ? G[0].x * (1.0f / 6.0f) : 0.f;
#pragma unroll
        for (int p = 0; p < 3; ++p) {
            const float* vp = v[(p + 1) % 3];
            const float* vm = v[(p + 2) % 3];
            const float c[3] = {vp[1] * vm[2] - vp[2] * vm[1], vp[2] * vm[0] - vp[0] * vm[2],
                                vp[0] * vm[1] - vp[1] * vm[0]};
            const float x[3] = {Q[1] * e[p][2] - Q[2] * e[p][1], Q[2] * e[p][0] - Q[0] * e[p][2],
                                Q[0] * e[p][1] - Q[1] * e[p][0]};
#pragma unroll
            for (int d = 0; d < 3; ++d) grad[p][d] = wf * (x[d] + g0 * c[d]) + V[p][d];   // V carries w_T through k.m_T
        }
    }
#pragma unroll
    for (int p = 0; p < 3; ++p)
#pragma unroll
        for (int d = 0; d < 3; ++d) corner[9 * (size_t)t + 3 * p + d] = grad[p][d];
}

// ---- A7: atomic-free scatter = gather over the vertex star through the CSR vertex->corner map (eq. 13) ------------
__global__ void dm_k_vertex_gather(const int32_t* __restrict__ csr_off, const int32_t* __restrict__ csr_corner,
                                   int n_vertices, const float* __restrict__ corner, float* __restrict__ dv)
{
    const int v = blockIdx.x * blockDim.x + threadIdx.x;
    if (v >= n_vertices) return;
    float a0 = 0.f, a1 = 0.f, a2 = 0.f;
    for (int j = csr_off[v]; j < csr_off[v + 1]; ++j) {
        const int c = csr_corner[j];  // = 3*face + corner
        a0 += corner[3 * (size_t)c];
        a1 += corner[3 * (size_t)c + 1];
        a2 += corner[3 * (size_t)c + 2];
    }
    dv[3 * (size_t)v] = a0;
    dv[3 * (size_t)v + 1] = a1;
    dv[3 * (size_t)v + 2] = a2;
}

// ---- surrounding stages: PSF multiply (and its adjoint) -----------------------------------------------------------
// c(k) = exp(-1/2 k^T Sigma k) e^{+i k.x0} / (h_x h_y h_z N_tot)   (eq. 2, 4; readings R5, R11);
// cuFFT transforms are unnormalised, so the 1/N_tot of the inverse DFT rides on c in both directions.
struct DmPsfDev {
    float cov[6];         // xx yy zz xy xz yz
    double org_turns[3];  // x0_a / L_a
    float inv_voxel;      // 1/(h_x h_y h_z N_tot): voxel scale and the 1/N_tot of the unnormalised cuFFT inverse
};
__device__ __forceinline__ cf dm_psf_coeff(const DmGridDev& grid, const DmPsfDev& psf, int ix, int iy, int iz)
{
    const int nx = dm_signed_freq(ix, grid.nx), ny = dm_signed_freq(iy, grid.ny), nz = iz;
    const float kx = grid.kstep[0] * nx, ky = grid.kstep[1] * ny, kz = grid.kstep[2] * nz;
    const float quad = psf.cov[0] * kx * kx + psf.cov[1] * ky * ky + psf.cov[2] * kz * kz +
                       2.0f * (psf.cov[3] * kx * ky + psf.cov[4] * kx * kz + psf.cov[5] * ky * kz);
    const float amp = expf(-0.5f * quad) * psf.inv_voxel;
    double tr = nx * psf.org_turns[0] + ny * psf.org_turns[1] + nz * psf.org_turns[2];
    tr -= rint(tr);
    float sn, cs;
    sincospif((float)(2.0 * tr), &sn, &cs);
    return {amp * cs, amp * sn};
}
// S = F c
__global__ void dm_k_psf_multiply(const float2* __restrict__ F, DmGridDev grid, DmPsfDev psf, float2* __restrict__ S)
{
    const long long n = (long long)grid.nx * grid.ny * grid.nzh;
    const long long l = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (l >= n) return;
    const int iz = (int)(l % grid.nzh), iy = (int)((l / grid.nzh) % grid.ny), ix = (int)(l / ((long long)grid.nzh * grid.ny));
    const cf c = dm_psf_coeff(grid, psf, ix, iy, iz);
    const float2 f = F[l];
    S[l] = make_float2(f.x * c.re - f.y * c.im, f.x * c.im + f.y * c.re);
}
// G = conj(c) w R,  w = 1 on n_z = 0 and n_z = N_z/2, else 2   (reading R14)
__global__ void dm_k_psf_adjoint(const float2* __restrict__ R, DmGridDev grid, DmPsfDev psf, float2* __restrict__ Gout)
{
    const long long n = (long long)grid.nx * grid.ny * grid.nzh;
    const long long l = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (l >= n) return;
    const int iz = (int)(l % grid.nzh), iy = (int)((l / grid.nzh) % grid.ny), ix = (int)(l / ((long long)grid.nzh * grid.ny));
    const cf c = dm_psf_coeff(grid, psf, ix, iy, iz);
    const float w = (iz == 0 || iz == grid.nz / 2) ? 1.0f : 2.0f;
    const float2 r = R[l];
    Gout[l] = make_float2(w * (r.x * c.re + r.y * c.im), w * (r.y * c.re - r.x * c.im));
}
// Drop Im on the planes n_z = 0 and n_z = N_z/2 after the (x,y) transforms: pins the half-spectrum inverse transform to
// numpy/pocketfft's irfftn semantics on a not-exactly-Hermitian spectrum (reading R13).
__global__ void dm_k_drop_selfconj_imag(float2* __restrict__ S, DmGridDev grid)
{
    const int l = blockIdx.x * blockDim.x + threadIdx.x;
    if (l >= grid.nx * grid.ny) return;
    S[(size_t)l * grid.nzh].y = 0.f;
    S[(size_t)l * grid.nzh + grid.nz / 2].y = 0.f;
}

// ---- PSF-parameter gradient (eq. 4 with reading R5) -----------------------------------------
// dL/dSigma_m = sum_k q_m(k) w Re( conj(R) F c ),  q = (-kx^2/2, -ky^2/2, -kz^2/2, -kx ky, -kx kz, -ky kz),
// R = rfft3(dL/dimage) (unnormalised; the 1/(N_tot h_x h_y h_z) rides on c), w as in dm_k_psf_adjoint.
// Two stages with fixed-order fp64 tree reductions (deterministic): DM_PSFG_BLOCKS block sums of 6 numbers, then one block.
#define DM_PSFG_BLOCKS 256
__global__ void __launch_bounds__(256)
dm_k_psf_grad_partial(const float2* __restrict__ R, const float2* __restrict__ F, DmGridDev grid, DmPsfDev psf,
                      double* __restrict__ partial)
{
    __shared__ double sh[6][256];
    const long long n = (long long)grid.nx * grid.ny * grid.nzh;
    double acc[6] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
    for (long long l = (long long)blockIdx.x * blockDim.x + threadIdx.x; l < n; l += (long long)gridDim.x * blockDim.x) {
        const int iz = (int)(l % grid.nzh), iy = (int)((l / grid.nzh) % grid.ny), ix = (int)(l / ((long long)grid.nzh * grid.ny));
        const cf c = dm_psf_coeff(grid, psf, ix, iy, iz);
        const float2 f = F[l], r = R[l];
        const float sre = f.x * c.re - f.y * c.im, sim = f.x * c.im + f.y * c.re;    // S = F c
        const float w = (iz == 0 || iz == grid.nz / 2) ? 1.0f : 2.0f;
        const double t = (double)(w * (r.x * sre + r.y * sim));                      // w Re(conj(R) S)
        const int nx = dm_signed_freq(ix, grid.nx), ny = dm_signed_freq(iy, grid.ny);
        const double kx = (double)(grid.kstep[0] * nx), ky = (double)(grid.kstep[1] * ny), kz = (double)(grid.kstep[2] * iz);
        acc[0] -= 0.5 * kx * kx * t;
        acc[1] -= 0.5 * ky * ky * t;
        acc[2] -= 0.5 * kz * kz * t;
        acc[3] -= kx * ky * t;
        acc[4] -= kx * kz * t;
        acc[5] -= ky * kz * t;
    }
#pragma unroll
    for (int m = 0; m < 6; ++m) sh[m][threadIdx.x] = acc[m];
    __syncthreads();
    for (int s = 128; s > 0; s >>= 1) {
        if (threadIdx.x < s)
#pragma unroll
            for (int m = 0; m < 6; ++m) sh[m][threadIdx.x] += sh[m][threadIdx.x + s];
        __syncthreads();
    }
    if (threadIdx.x < 6) partial[6 * blockIdx.x + threadIdx.x] = sh[threadIdx.x][0];
}
__global__ void __launch_bounds__(DM_PSFG_BLOCKS)
dm_k_psf_grad_final(const double* __restrict__ partial, float* __restrict__ out6)
{
    __shared__ double sh[6][DM_PSFG_BLOCKS];
#pragma unroll
    for (int m = 0; m < 6; ++m) sh[m][threadIdx.x] = partial[6 * threadIdx.x + m];
    __syncthreads();
    for (int s = DM_PSFG_BLOCKS / 2; s > 0; s >>= 1) {
        if (threadIdx.x < s)
#pragma unroll
            for (int m = 0; m < 6; ++m) sh[m][threadIdx.x] += sh[m][threadIdx.x + s];
        __syncthreads();
    }
    if (threadIdx.x < 6) out6[threadIdx.x] = (float)sh[threadIdx.x][0];
}

// ---- narrow band: the in-band interval [z_lo, z_hi) of every (i_x, i_y) row ----------------------
// (the band is convex, so the in-band frequencies of a row are contiguous; an empty row gets z_lo = z_hi = 0)
__global__ void dm_k_band_rows(DmGridDev grid, int2* __restrict__ band_z)
{
    const int row = blockIdx.x * blockDim.x + threadIdx.x;
    if (row >= grid.nx * grid.ny) return;
    const int nx = dm_signed_freq(row / grid.ny, grid.nx), ny = dm_signed_freq(row % grid.ny, grid.ny);
    int lo = 0, hi = 0;
    bool any = false;
    for (int iz = 0; iz < grid.nzh; ++iz)
        if (dm_in_band(grid, nx, ny, iz)) {
            if (!any) lo = iz;
            any = true;
            hi = iz + 1;
        }
    band_z[row] = make_int2(lo, hi);
}

// ---- area-normalised membrane density (eq. 12-13) -----------------------------------------------------
// u = F / |Lambda|: scale the spectrum by the fp64 total area the k = 0 kernels left in *total
__global__ void dm_k_scale_spectrum(float2* __restrict__ F, long long n, const double* __restrict__ total)
{
    const long long l = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (l >= n) return;
    const float inv = (float)(1.0 / *total);
    float2 f = F[l];
    f.x *= inv;
    f.y *= inv;
    F[l] = f;
}
// sdot = sum_k Re(conj(G) F) over the stored entries, fp64, two fixed-order stages
#define DM_DOT_BLOCKS 256
__global__ void __launch_bounds__(256)
dm_k_dot_partial(const float2* __restrict__ G, const float2* __restrict__ F, long long n, double* __restrict__ partial)
{
    __shared__ double sh[256];
    double acc = 0.0;
    for (long long l = (long long)blockIdx.x * blockDim.x + threadIdx.x; l < n; l += (long long)gridDim.x * blockDim.x) {
        const float2 g = G[l], f = F[l];
        acc += (double)g.x * (double)f.x + (double)g.y * (double)f.y;
    }
    sh[threadIdx.x] = acc;
    __syncthreads();
    for (int s = 128; s > 0; s >>= 1) {
        if (threadIdx.x < s) sh[threadIdx.x] += sh[threadIdx.x + s];
        __syncthreads();
    }
    if (threadIdx.x == 0) partial[blockIdx.x] = sh[0];
}
__global__ void __launch_bounds__(DM_DOT_BLOCKS)
dm_k_dot_final(const double* __restrict__ partial, double* __restrict__ out)
{
    __shared__ double sh[DM_DOT_BLOCKS];
    sh[threadIdx.x] = partial[threadIdx.x];
    __syncthreads();
    for (int s = DM_DOT_BLOCKS / 2; s > 0; s >>= 1) {
        if (threadIdx.x < s) sh[threadIdx.x] += sh[threadIdx.x + s];
        __syncthreads();
    }
    if (threadIdx.x == 0) *out = sh[0];
}
