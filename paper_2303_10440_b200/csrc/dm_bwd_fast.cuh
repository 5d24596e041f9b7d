// dm_bwd_fast.cuh -- optimised backward mesh-FT kernel (rows A1, A6 of the hot path), sm_100a.
//
// Layout.  One THREAD owns one triangle and keeps its 13 k-sums in registers; one WARP owns a compact patch of 32
// triangles (dm_patches.h) and a CTA of four warps walks a range of (i_x,i_y) rows of the stored spectrum, innermost
// along z.  Every thread of the CTA is at the SAME frequency at the same time, so everything that depends on k only --
// kappa = conj(G) (surface) or i conj(G)/|k|^2 (volume), k_z -- is computed once per CTA and row into shared memory and
// read back as one broadcast LDS.128 per pair, and there is no reduction across threads at all (O(N n_v)
// backward; :182-186 eq. 13 is the later CSR gather).
//
// Shared vertex phases (north_star: "each vertex's phase e^{-ik.v} is computed once per (k-tile, vertex) and reused across
// its incident triangles").  A patch of 32 triangles has about 28 distinct vertices.  Lane l owns vertex slot l of its
// patch: per frequency it advances that ONE phase by a
// complex rotation, multiplies it by kappa and stores A_v = kappa e^{-ik.v} in shared memory; after a __syncwarp the 32
// triangle lanes read the A_v of their three corners.  Per pair this is 8 FP32 operations + 1 STS + 3 LDS instead of the
// 24 operations of three private phases.
//
// Arithmetic of the generic pair.  With nodes x_j = k.v_j, E_j = e^{-i x_j} and gaps
// p = x_1-x_0, q = x_2-x_0, r = q-p, eq. 9 is  g = sum_j c_j E_j  with REAL coefficients
//     c_0 = -1/(pq),  c_1 = 1/(pr),  c_2 = -1/(qr)        (one MUFU.RCP of pqr),
// and its node derivatives (the closed form of PAPER.md:171-173 eq. 11 with reading R2, regrouped) are
//     dg/dx_1 = sum_j al_j E_j - i c_1 E_1,   al_0 = q c_0^2, al_2 = -q c_2^2, al_1 = -al_0-al_2   (sum_j c_j = 0)
//     dg/dx_2 = sum_j be_j E_j - i c_2 E_2,   be_0 = p c_0^2, be_1 = -p c_1^2, be_2 = -be_0-be_1
//     dg/dx_0 = -i g - dg/dx_1 - dg/dx_2.
// With A_j = kappa E_j the four real numbers a pair contributes are
//     s0 = Re(kappa g) = sum c_j Re A_j,  sI = Im(kappa g) = sum c_j Im A_j,
//     sb = Re(kappa dg/dx_1) = sum al_j Re A_j + c_1 Im A_1,   sc likewise,
// all taken on differences of the A_j (every coefficient triple sums to zero).
// Phases advance along z by one complex rotation (rotor e^{-i kstep_z v_z} built in fp64 by the geometry pre-pass) and
// are re-seeded every SEG (8, 16 or 32) frequencies from exact values: the exact row phase (32-bit integer turns) times a
// row-independent table of exact z-phases kept in shared memory.
//
// Near-degenerate pairs (reading R4).  The derivative coefficients grow like 1/(gap^2 gap'), so a pair
// with  m1^2 m2 <= tau_b  (m1 <= m2 the two smallest |gaps|)  is excluded from the fast sums (its reciprocal is forced to 0) and flagged in a per-
// thread bit mask.  After each chunk of <= DM_BF_CHUNK frequencies the WARP pools its flagged pairs in shared memory,
// sorted by owner, and evaluates them 32 at a time, one pair per lane whatever its owner: the series branch where all
// gaps are small, the branch-free far-pair variant otherwise.  A segmented warp scan sums the results of one owner and
// the run's last lane adds them to that owner's shared accumulators -- a fixed order, so the result is bitwise
// reproducible (reading R22), and the divergent work is spread evenly over the lanes.
#pragma once
#include "dm_kernels.cuh"
#include "dm_patches.h"

#ifndef DM_BF_THREADS
#define DM_BF_THREADS 128
#endif
#ifndef DM_BF_MINCTA
#define DM_BF_MINCTA 5         // resident CTAs per SM the register allocation aims at (<= 102 registers)
#endif
#define DM_BF_SEG 32            // bits of one flag word
#define DM_BF_UNR 8             // unroll of the fast loop
#ifndef DM_BF_STAGE
#define DM_BF_STAGE 8           // frequencies whose vertex phases are staged in shared memory at a time (divides DM_BF_UNR)
#endif
#define DM_BF_TREC 4            // float4 per triangle record
#define DM_BF_VREC 2            // float4 per vertex-slot record

// device copies of the patch tables (topology; built at plan creation)
struct DmPatchDev {
    const int32_t* face;    // [n_lanes]       face of lane, -1 = idle
    const int32_t* vid;     // [n_lanes]       vertex of slot l of the patch, -1 = unused
    const uint32_t* loc;    // [n_lanes]       corner slots l0 | l1 << 8 | l2 << 16
    int n_lanes;            // 32 * number of patches, a multiple of DM_BF_THREADS
};

// Records rebuilt every call (row A1), indexed by lane i = 32 * patch + l:
//   triangle  trec[4i..4i+3] = (u_0.xyz [uint32 bit patterns: v_0 / L in fixed-point turns], loc bits)
//                              (eb.xyz, longest squared edge)   (ec.xyz, -)   (m_T.xyz, |m_T|)       eb = v_1-v_0, ec = v_2-v_0
//   vertex    vrec[2i..2i+1] (slot l of the patch):  (u.xyz turns, rho.re)  (rho.im, -, -, -),  rho = e^{-i kstep_z v_z}
__global__ void dm_k_bwd_geometry(const float* __restrict__ vertices, const int32_t* __restrict__ faces, DmPatchDev pt,
                                  DmGridDev grid, float4* __restrict__ trec, float4* __restrict__ vrec,
                                  unsigned int* __restrict__ hmax2_bits)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= pt.n_lanes) return;   // n_lanes is a multiple of the warp size: whole warps leave
    float h2 = 0.f, e2sum = 0.f;
    {
        int f = pt.face[i];
        if (f < 0) f = pt.face[i & ~31];   // idle lane: any valid triangle of the patch (lane 0 holds one)
        if (f < 0) f = 0;                  // padding patch
        float v[3][3];
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            const int iv = faces[3 * f + j];
#pragma unroll
            for (int d = 0; d < 3; ++d) v[j][d] = vertices[3 * iv + d];
        }
        uint32_t u[3];
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            double tt = (double)v[0][d] * grid.inv_len[d];
            tt -= floor(tt);
            u[d] = (uint32_t)(unsigned long long)(tt * 4294967296.0 + 0.5);
        }
        const float eb[3] = {v[1][0] - v[0][0], v[1][1] - v[0][1], v[1][2] - v[0][2]};
        const float ec[3] = {v[2][0] - v[0][0], v[2][1] - v[0][1], v[2][2] - v[0][2]};
        float m[3];
        dm_cross(eb, ec, m);
        // edge statistics of the mesh (they scale the flag threshold)
        const float ed[3] = {ec[0] - eb[0], ec[1] - eb[1], ec[2] - eb[2]};
        const float a2 = eb[0] * eb[0] + eb[1] * eb[1] + eb[2] * eb[2], b2 = ec[0] * ec[0] + ec[1] * ec[1] + ec[2] * ec[2],
                    c2 = ed[0] * ed[0] + ed[1] * ed[1] + ed[2] * ed[2];
        if (pt.face[i] >= 0) {
            h2 = fmaxf(fmaxf(a2, b2), c2);
            e2sum = a2 + b2 + c2;
        }
        const float wf = grid.face_w ? grid.face_w[f] : 1.0f;   // density weight of the face
        const float mn = wf * sqrtf(m[0] * m[0] + m[1] * m[1] + m[2] * m[2]);
        m[0] *= wf, m[1] *= wf, m[2] *= wf;
        float4* o = trec + (size_t)DM_BF_TREC * i;
        o[0] = make_float4(__uint_as_float(u[0]), __uint_as_float(u[1]), __uint_as_float(u[2]), __uint_as_float(pt.loc[i]));
        o[1] = make_float4(eb[0], eb[1], eb[2], fmaxf(fmaxf(a2, b2), c2));
        o[2] = make_float4(ec[0], ec[1], ec[2], 0.f);
        o[3] = make_float4(m[0], m[1], m[2], mn);
    }
    {
        const size_t s = (size_t)i;
        const int iv = pt.vid[s];
        float4 a = make_float4(0.f, 0.f, 0.f, 1.f), b = make_float4(0.f, 0.f, 0.f, 0.f);
        if (iv >= 0) {
            uint32_t u[3];
#pragma unroll
            for (int d = 0; d < 3; ++d) {
                double tt = (double)vertices[3 * iv + d] * grid.inv_len[d];
                tt -= floor(tt);
                u[d] = (uint32_t)(unsigned long long)(tt * 4294967296.0 + 0.5);
            }
            double tz = (double)vertices[3 * iv + 2] * grid.inv_len[2];
            tz -= rint(tz);
            double sn, cs;
            sincospi(2.0 * tz, &sn, &cs);
            a = make_float4(__uint_as_float(u[0]), __uint_as_float(u[1]), __uint_as_float(u[2]), (float)cs);
            b.x = (float)(-sn);
        }
        vrec[DM_BF_VREC * s] = a;
        vrec[DM_BF_VREC * s + 1] = b;
    }
    dm_edge_stats_add(hmax2_bits, h2, e2sum, grid.edge_fix);
}

// shared-memory queue of one warp's flagged pairs of one chunk
#define DM_BF_CHUNK 96          // frequencies per chunk = 3 flag words per thread
struct DmBfQueue {
    unsigned char code[32 * DM_BF_CHUNK];  // frequency index inside the chunk, in (owner lane, frequency) order; the
                                           // owner of entry e is found from the lanes' prefix sums
};

// what one pair adds to the row sums (plain and k_z-weighted sums of s0, sI, sb, sc)
struct DmBfRow {
    float S0, S0z, SI, SIz, SB, SBz, SC, SCz;
};
template <int MODE>
__device__ __forceinline__ void dm_bf_add(DmBfRow& a, float kz, float om, float s0, float sI, float sb, float sc)
{
    if (MODE == 0) {  // volume: omega = k.m_T weights the derivative sums, Q needs k s0
        sI *= om;
        sb *= om;
        sc *= om;
        a.S0z = fmaf(kz, s0, a.S0z);
    }
    a.S0 += s0;
    a.SI += sI;
    a.SIz = fmaf(kz, sI, a.SIz);
    a.SB += sb;
    a.SBz = fmaf(kz, sb, a.SBz);
    a.SC += sc;
    a.SCz = fmaf(kz, sc, a.SCz);
}

// The fast evaluation of ONE pair (generic closed form) from the staged A_j = kappa e^{-i x_j} of its three corners;
// returns true when the pair is excluded (flagged) instead.
template <int MODE>
__device__ __forceinline__ bool dm_bf_pair(const float kz, const cf A0, const cf A1, const cf A2, const float prow,
                                           const float qrow, const float omrow, const float ebz, const float ecz,
                                           const float mz, const float tau_k, DmBfRow& rs)
{
    const float p = fmaf(kz, ebz, prow), q = fmaf(kz, ecz, qrow), r = q - p;
    const float pqr = (p * q) * r;
    // the largest derivative coefficient is 1/(m1^2 m2), m1 <= m2 <= m3 the sorted |gaps| (m3 = m1 + m2 always): the pair
    // leaves the fast path when m1^2 m2 = m1 |pqr| / m3 <= tau_k  (also catches p = q = r = 0); tau_k = the threshold of
    // this triangle on this row (tau_b, larger for a triangle that is coarse for the grid)
    const float m1 = fminf(fminf(fabsf(p), fabsf(q)), fabsf(r));
    const float m3 = fmaxf(fmaxf(fabsf(p), fabsf(q)), fabsf(r));
    const bool bad = !(m1 * fabsf(pqr) > tau_k * m3);
    const float R = bad ? 0.f : dm_rcp_approx(pqr);
    const float c0 = -r * R, c1 = q * R, c2 = -p * R;
    const float c0s = c0 * c0, c1s = c1 * c1, c2s = c2 * c2;
    const float a0 = q * c0s, a2 = -q * c2s;      // al_1 = -al_0 - al_2
    const float b0 = p * c0s, nb1 = p * c1s;      // be_1 = -nb1, be_2 = -be_0 - be_1
    const float d01r = A0.re - A1.re, d21r = A2.re - A1.re, d02r = d01r - d21r;
    const float d01i = A0.im - A1.im, d21i = A2.im - A1.im;
    const float s0 = fmaf(c0, d01r, c2 * d21r);
    const float sI = fmaf(c0, d01i, c2 * d21i);
    const float sb = fmaf(a0, d01r, fmaf(a2, d21r, c1 * A1.im));
    const float sc = fmaf(b0, d02r, fmaf(nb1, d21r, c2 * A2.im));
    dm_bf_add<MODE>(rs, kz, fmaf(kz, mz, omrow), s0, sI, sb, sc);
    return bad;
}

// ---- A6 backward, fast kernel -----------------------------------------------------------------------------------
// grid = (n_lanes / DM_BF_THREADS, n_split): one warp per patch; part[(split*13 + s)*n_faces + face] as in
// dm_k_backward_robust.  BAND = the narrow band is set (band_z holds the in-band z interval of every row).
// SEG = frequencies between exact phase seeds (8, 16 or 32; chosen by the host so that the seed
// table fits).  Dynamic shared memory:
//   2 * nzh float4                      double-buffered rows (kappa.re, kappa.im, k_z, -)
//   (nseg-1) * 128 float2               seed table ztab[a-1][tid] = e^{-2 pi i (a SEG) u_z} of the thread's vertex
//                                       slot, a = 1 .. nseg-1, nseg = ceil(nzh/SEG): with the exact row phase
//                                       e^{-2 pi i (n_x u_x + n_y u_y)} (integer turns, one accurate sincospi per row) a
//                                       phase is never more than SEG-1 fp32 rotations away from an exact value
//   4 * DM_BF_STAGE * 32 float2         per warp: A_v = kappa e^{-ik.v} of the patch's vertex slots for DM_BF_STAGE
//                                       consecutive frequencies
template <int MODE, int SEG, bool BAND>
__global__ void __launch_bounds__(DM_BF_THREADS, DM_BF_MINCTA)
dm_k_backward_fast(const float4* __restrict__ trec_g, const float4* __restrict__ vrec_g, DmPatchDev pt, int n_faces,
                   DmGridDev grid, int ix_begin, int ix_end, int rows_per_split, float tau_b,
                   const float2* __restrict__ G, const int2* __restrict__ band_z, float* __restrict__ part)
{
    static_assert(SEG == 8 || SEG == 16 || SEG == 32, "SEG divides the 32-bit flag word");
    static_assert(DM_BF_UNR % DM_BF_STAGE == 0 && SEG % DM_BF_UNR == 0, "stages tile the unrolled body, bodies tile a segment");
    extern __shared__ float4 dm_bf_smem[];
    __shared__ DmBfQueue queue[DM_BF_THREADS / 32];
    __shared__ float4 trec[DM_BF_THREADS * DM_BF_TREC];    // this CTA's triangle records (the pooled path reads other lanes')
    __shared__ float wacc[(DM_BF_THREADS / 32) * 8 * 32];  // per warp: 8 row sums x 32 owners, filled by the pooled path
    float4* const sk = dm_bf_smem;
    const int tid = threadIdx.x, lane = tid & 31, wrp = tid >> 5;
    const int gl = blockIdx.x * DM_BF_THREADS + tid;       // global lane = 32 * patch + lane
    const int face = pt.face[gl];
    const bool live = face >= 0;
    const float4 r0 = trec_g[(size_t)DM_BF_TREC * gl], r3 = trec_g[(size_t)DM_BF_TREC * gl + 1],
                 r4 = trec_g[(size_t)DM_BF_TREC * gl + 2], r5 = trec_g[(size_t)DM_BF_TREC * gl + 3];
    trec[tid * DM_BF_TREC + 0] = r0;
    trec[tid * DM_BF_TREC + 1] = r3;
    trec[tid * DM_BF_TREC + 2] = r4;
    trec[tid * DM_BF_TREC + 3] = r5;
    const uint32_t loc = __float_as_uint(r0.w);
    const int l0 = (int)(loc & 255u), l1 = (int)((loc >> 8) & 255u), l2 = (int)((loc >> 16) & 255u);
    // the vertex slot this lane owns (slot lane of its patch)
    const float4 va0 = vrec_g[(size_t)DM_BF_VREC * gl], va1 = vrec_g[(size_t)DM_BF_VREC * gl + 1];
    const uint32_t uax = __float_as_uint(va0.x), uay = __float_as_uint(va0.y), uaz = __float_as_uint(va0.z);
    const cf rhoa = {va0.w, va1.x};
    const int nzh = grid.nzh;
    const int n_rows = (ix_end - ix_begin) * grid.ny;
    const int row_begin = blockIdx.y * rows_per_split;
    const int row_end = min(n_rows, row_begin + rows_per_split);
    DmBfQueue& Q = queue[wrp];
    const float4* const wrec = trec + wrp * 32 * DM_BF_TREC;   // records of this warp's 32 triangles

    // seed table (row-independent): exact z-phases of this thread's vertex slots at every multiple of SEG
    const int nseg = (nzh + SEG - 1) / SEG;
    float2* const ztab = reinterpret_cast<float2*>(dm_bf_smem + 2 * nzh);
    float2* const at = ztab + (size_t)(nseg - 1) * DM_BF_THREADS + wrp * DM_BF_STAGE * DM_PATCH_MAXV;
    for (int a = 1; a < nseg; ++a) {
        const uint32_t za = (uint32_t)(a * SEG);
        const cf z0 = dm_expmi_turns(za * uaz);
        ztab[(a - 1) * DM_BF_THREADS + tid] = make_float2(z0.re, z0.im);
    }

#pragma unroll
    for (int i = 0; i < 8; ++i) wacc[i * DM_BF_THREADS + tid] = 0.f;
    // acc: [0] S0 | [1..3] Q | [4..6] W | [7..9] Vb | [10..12] Vc   (dm_k_backward_robust)
    float acc[DM_BWD_NSUM];
#pragma unroll
    for (int s = 0; s < DM_BWD_NSUM; ++s) acc[s] = 0.f;

    // stage kappa and k_z of one row into buffer b
    auto stage_row = [&](int row, int b) {
        const int ix = ix_begin + row / grid.ny, iy = row % grid.ny;
        const int nx = dm_signed_freq(ix, grid.nx), ny = dm_signed_freq(iy, grid.ny);
        const float kx = grid.kstep[0] * nx, ky = grid.kstep[1] * ny;
        const float2* Grow = G + ((size_t)ix * grid.ny + iy) * nzh;
        for (int iz = tid; iz < nzh; iz += DM_BF_THREADS) {
            const float kz = grid.kstep[2] * iz;
            float2 Gk = Grow[iz];
            if (BAND && !dm_in_band(grid, nx, ny, iz)) Gk = make_float2(0.f, 0.f);  // narrow band: the cotangent outside is ignored
            float4 o;
            if (MODE == 1) {
                o = make_float4(Gk.x, -Gk.y, kz, 0.f);                       // conj(G)
            } else {
                const float k2 = kx * kx + ky * ky + kz * kz;
                const float inv_k2 = (k2 > 0.f) ? 1.0f / k2 : 0.f;           // k = 0 is handled by dm_k_corner_grads
                o = make_float4(Gk.y * inv_k2, Gk.x * inv_k2, kz, 0.f);      // i conj(G) / |k|^2
            }
            sk[b * nzh + iz] = o;
        }
    };

    // one stage of n <= DM_BF_STAGE frequencies starting at z: every lane writes A_v of its vertex slot(s), then every
    // lane evaluates its triangle at those frequencies; returns the flags of the stage (bit j = frequency z + j)
    auto run_stage = [&](const float4* skr, int z, int n, bool full, cf& Ea, float prow, float qrow, float omrow,
                         float tau_row, DmBfRow& rs) -> uint32_t {
        if (full) {
#pragma unroll
            for (int j = 0; j < DM_BF_STAGE; ++j) {
                const float4 kk = skr[z + j];
                const cf A = cmul(cf{kk.x, kk.y}, Ea);
                at[j * DM_PATCH_MAXV + lane] = make_float2(A.re, A.im);
                Ea = cmul(Ea, rhoa);
            }
        } else {
#pragma unroll 1
            for (int j = 0; j < n; ++j) {
                const float4 kk = skr[z + j];
                const cf A = cmul(cf{kk.x, kk.y}, Ea);
                at[j * DM_PATCH_MAXV + lane] = make_float2(A.re, A.im);
                Ea = cmul(Ea, rhoa);
            }
        }
        __syncwarp();
        uint32_t sf = 0;
        if (full) {
#pragma unroll
            for (int j = 0; j < DM_BF_STAGE; ++j) {
                const float kz = skr[z + j].z;
                const float2 a0 = at[j * DM_PATCH_MAXV + l0], a1 = at[j * DM_PATCH_MAXV + l1], a2 = at[j * DM_PATCH_MAXV + l2];
                if (dm_bf_pair<MODE>(kz, cf{a0.x, a0.y}, cf{a1.x, a1.y}, cf{a2.x, a2.y}, prow, qrow, omrow, r3.z, r4.z, r5.z,
                                     tau_row, rs))
                    sf |= 1u << j;
            }
        } else {
#pragma unroll 1
            for (int j = 0; j < n; ++j) {
                const float kz = skr[z + j].z;
                const float2 a0 = at[j * DM_PATCH_MAXV + l0], a1 = at[j * DM_PATCH_MAXV + l1], a2 = at[j * DM_PATCH_MAXV + l2];
                if (dm_bf_pair<MODE>(kz, cf{a0.x, a0.y}, cf{a1.x, a1.y}, cf{a2.x, a2.y}, prow, qrow, omrow, r3.z, r4.z, r5.z,
                                     tau_row, rs))
                    sf |= 1u << j;
            }
        }
        __syncwarp();
        return sf;
    };

    if (row_begin < row_end) stage_row(row_begin, 0);
    __syncthreads();
    for (int row = row_begin; row < row_end; ++row) {
        const int b = (row - row_begin) & 1;
        if (row + 1 < row_end) stage_row(row + 1, b ^ 1);
        const float4* __restrict__ skr = sk + b * nzh;
        const int ix = ix_begin + row / grid.ny, iy = row % grid.ny;
        const int nx = dm_signed_freq(ix, grid.nx), ny = dm_signed_freq(iy, grid.ny);
        const float kx = grid.kstep[0] * nx, ky = grid.kstep[1] * ny;
        const float prow = fmaf(kx, r3.x, ky * r3.y), qrow = fmaf(kx, r4.x, ky * r4.y);
        const float omrow = fmaf(kx, r5.x, ky * r5.y);
        // flag threshold of this triangle on this row: tau_b max(1, (|k| h_T / 12)^3), |k| the largest of the row, h_T the
        // longest edge of the triangle.  On a triangle that is large for the grid (|k| h >> 1) the rounding error of a gap
        // k.e grows like |k| h while the integral decays like 1/(|k| h)^2; the factor is exactly 1 when |k| h_T <= 12
        const float kzm = grid.kstep[2] * (float)(nzh - 1);
        const float kh2 = (1.0f / 144.0f) * (kx * kx + ky * ky + kzm * kzm) * trec[tid * DM_BF_TREC + 1].w;   // (re-read: one register less)
        const float tau_row = tau_b * fmaxf(1.0f, kh2 * sqrtf(kh2));
        // exact row phase e^{-i (k_x v_x + k_y v_y)} of the lane's vertex slot
        const cf Xa = dm_expmi_turns((uint32_t)nx * uax + (uint32_t)ny * uay);
        DmBfRow rs = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};

        // narrow band: only the in-band interval of the row, started at a seed position
        int z_lo = 0, z_hi = nzh;
        if (BAND) {
            const int2 bz = band_z[ix * grid.ny + iy];
            z_lo = bz.x & ~(SEG - 1);
            z_hi = bz.y;
        }
        for (int zc = z_lo; zc < z_hi; zc += DM_BF_CHUNK) {
            const int clen = min(DM_BF_CHUNK, z_hi - zc);
            uint32_t fl[DM_BF_CHUNK / 32];
            // ---- fast pass over the chunk: bodies of DM_BF_UNR frequencies, exact seeds every SEG ---------------------
            cf Ea = Xa;
#pragma unroll
            for (int w = 0; w < DM_BF_CHUNK / 32; ++w) {
                uint32_t word = 0;
                const int wbeg = zc + 32 * w;
                const int wlen = min(32, zc + clen - wbeg);
                if (wlen > 0) {
                    const int nfull = wlen / DM_BF_UNR;
                    int z0 = wbeg;
#pragma unroll 1
                    for (int s = 0; s <= nfull; ++s, z0 += DM_BF_UNR) {
                        const int len = (s < nfull) ? DM_BF_UNR : wlen - nfull * DM_BF_UNR;
                        if (len == 0) break;
                        if ((z0 & (SEG - 1)) == 0) {   // exact seed
                            Ea = Xa;
                            if (z0 > 0) {
                                const float2 a0 = ztab[(size_t)(z0 / SEG - 1) * DM_BF_THREADS + tid];
                                Ea = cmul(Xa, cf{a0.x, a0.y});
                            }
                        }
                        uint32_t sf = 0;
                        if (len == DM_BF_UNR) {
#pragma unroll
                            for (int h = 0; h < DM_BF_UNR / DM_BF_STAGE; ++h)
                                sf |= run_stage(skr, z0 + h * DM_BF_STAGE, DM_BF_STAGE, true, Ea, prow, qrow, omrow, tau_row, rs)
                                      << (h * DM_BF_STAGE);
                        } else {
#pragma unroll 1
                            for (int j0 = 0; j0 < len; j0 += DM_BF_STAGE)
                                sf |= run_stage(skr, z0 + j0, min(DM_BF_STAGE, len - j0), false, Ea, prow, qrow, omrow, tau_row, rs) << j0;
                        }
                        word |= sf << (s * DM_BF_UNR);
                    }
                }
                fl[w] = live ? word : 0u;
            }
            // ---- pooled slow path -------------------------------------------------------------------------------------
            int cnt = 0;
#pragma unroll
            for (int sg = 0; sg < DM_BF_CHUNK / DM_BF_SEG; ++sg) cnt += __popc(fl[sg]);
            if (__any_sync(0xffffffffu, cnt != 0)) {
                int off = cnt;  // inclusive prefix sum over lanes
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    const int n = __shfl_up_sync(0xffffffffu, off, o);
                    if (lane >= o) off += n;
                }
                const int total = __shfl_sync(0xffffffffu, off, 31);
                // owners queue their pairs in (lane, frequency) order
                int w = off - cnt;
#pragma unroll
                for (int sg = 0; sg < DM_BF_CHUNK / DM_BF_SEG; ++sg) {
                    uint32_t f = fl[sg];
                    while (f) {
                        const int j = __ffs(f) - 1;
                        f &= f - 1;
                        Q.code[w++] = (unsigned char)(sg * DM_BF_SEG + j);
                    }
                }
                __syncwarp();
                // rounds of 32 queued pairs: every lane evaluates one pair; a segmented scan over the (sorted) owners sums
                // the pairs of one owner, and the last lane of each run adds the run into the owner's shared accumulators
                for (int base = 0; base < total; base += 32) {
                    const int e = base + lane;
                    const bool have = e < total;
                    // owner of entry e = number of lanes whose inclusive prefix sum is <= e (binary search by shuffles)
                    int own = 0;
#pragma unroll
                    for (int st = 16; st > 0; st >>= 1) {
                        const int v = __shfl_sync(0xffffffffu, off, own + st - 1);
                        if (v <= e) own += st;
                    }
                    own = have ? own : 0;
                    const int ol = have ? own : -1 - lane, jz = zc + (have ? (int)Q.code[e] : 0);
                    const float4* orc = wrec + own * 4;
                    const float4 q0 = orc[0], q3 = orc[1], q4 = orc[2], q5 = orc[3];
                    const float4 kk = skr[jz];
                    const float kz = kk.z;
                    const float p = fmaf(kz, q3.z, fmaf(kx, q3.x, ky * q3.y));
                    const float q = fmaf(kz, q4.z, fmaf(kx, q4.x, ky * q4.y));
                    const bool series = fmaxf(fmaxf(fabsf(p), fabsf(q)), fabsf(q - p)) < DM_SERIES_RADIUS;
                    cf psi = {0.f, 0.f}, dp = {0.f, 0.f}, dq = {0.f, 0.f};
                    if (__any_sync(0xffffffffu, have && series)) {
                        cf a, b, c;
                        dm_psi_series<true>(series ? p : 0.f, series ? q : 0.f, a, b, c);
                        if (series) { psi = a; dp = b; dq = c; }
                    }
                    if (__any_sync(0xffffffffu, have && !series)) {
                        cf a, b, c;
                        dm_psi_far_uniform(series ? 0.f : p, series ? 1.f : q, a, b, c);
                        if (!series) { psi = a; dp = b; dq = c; }
                    }
                    const cf E = dm_expmi_turns_fast(dm_phase_turns(nx, ny, jz, __float_as_uint(q0.x), __float_as_uint(q0.y),
                                                                    __float_as_uint(q0.z)));
                    const cf kE = cmul(cf{kk.x, kk.y}, E);
                    const cf kg = cmul(kE, psi);
                    DmBfRow v = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
                    if (have)
                        dm_bf_add<MODE>(v, kz, fmaf(kz, q5.z, fmaf(kx, q5.x, ky * q5.y)), kg.re, kg.im,
                                        kE.re * dp.re - kE.im * dp.im, kE.re * dq.re - kE.im * dq.im);
                    float vv[8] = {v.S0, v.S0z, v.SI, v.SIz, v.SB, v.SBz, v.SC, v.SCz};
#pragma unroll
                    for (int o = 1; o < 32; o <<= 1) {
                        const int ko = __shfl_up_sync(0xffffffffu, ol, o);
                        const bool take = lane >= o && ko == ol;
#pragma unroll
                        for (int i = 0; i < 8; ++i) {
                            if (MODE == 1 && i == 1) continue;  // S0z is a volume-mode sum
                            const float x = __shfl_up_sync(0xffffffffu, vv[i], o);
                            if (take) vv[i] += x;
                        }
                    }
                    const int kn = __shfl_down_sync(0xffffffffu, ol, 1);
                    if (have && (lane == 31 || kn != ol)) {
#pragma unroll
                        for (int i = 0; i < 8; ++i) {
                            if (MODE == 1 && i == 1) continue;
                            wacc[(wrp * 8 + i) * 32 + ol] += vv[i];
                        }
                    }
                    __syncwarp();
                }
                // owners take their sums back (and clear them)
                if (cnt != 0) {
                    float* a = wacc + wrp * 8 * 32 + lane;
                    rs.S0 += a[0];
                    if (MODE == 0) rs.S0z += a[32];
                    rs.SI += a[64];
                    rs.SIz += a[96];
                    rs.SB += a[128];
                    rs.SBz += a[160];
                    rs.SC += a[192];
                    rs.SCz += a[224];
#pragma unroll
                    for (int i = 0; i < 8; ++i) a[32 * i] = 0.f;
                }
                __syncwarp();
            }
        }
        // fold the row into the 13 sums
        if (MODE == 1) {
            acc[0] += rs.S0;
        } else {
            acc[1] = fmaf(kx, rs.S0, acc[1]);
            acc[2] = fmaf(ky, rs.S0, acc[2]);
            acc[3] += rs.S0z;
        }
        acc[4] = fmaf(kx, rs.SI, acc[4]);
        acc[5] = fmaf(ky, rs.SI, acc[5]);
        acc[6] += rs.SIz;
        acc[7] = fmaf(kx, rs.SB, acc[7]);
        acc[8] = fmaf(ky, rs.SB, acc[8]);
        acc[9] += rs.SBz;
        acc[10] = fmaf(kx, rs.SC, acc[10]);
        acc[11] = fmaf(ky, rs.SC, acc[11]);
        acc[12] += rs.SCz;
        __syncthreads();  // next row's buffer is complete; this row's buffer may be overwritten
    }
    if (live) {
#pragma unroll
        for (int s = 0; s < DM_BWD_NSUM; ++s) part[((size_t)blockIdx.y * DM_BWD_NSUM + s) * n_faces + face] = acc[s];
    }
}
