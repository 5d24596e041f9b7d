// dm_bwd_fast.cuh -- optimised backward mesh-FT kernel (rows A1, A6 of the hot path), sm_100a.
//
// Layout.  One THREAD owns one triangle and keeps its 13 k-sums in registers; one WARP owns a compact patch of 32
// triangles (dm_patches.h) and walks a range of (i_x,i_y) rows of the stored spectrum, innermost along z.  The warps of a
// CTA are completely independent -- there is no CTA-wide barrier after the set-up: everything that depends on k only
// (kappa = conj(G) [surface] or i conj(G)/|k|^2 [volume], zero outside the narrow band) is written once per call by the
// elementwise pre-pass dm_k_kappa, and every warp stages the 32 frequencies it is about to visit from that array into its
// own 256 bytes of shared memory (one coalesced load per lane, prefetched one chunk ahead).  There is no reduction across
// threads at all (O(N n_v) backward; :182-186 eq. 13 is the later CSR gather).
//
// Shared vertex phases (north_star: "each vertex's phase e^{-ik.v} is computed once per (k-tile, vertex) and reused across
// its incident triangles").  A patch of 32 triangles has about 28 distinct vertices.  Lane l owns vertex slot l of its
// patch: per frequency it advances that ONE phase by a complex rotation, multiplies it by kappa and stores
// A_v = kappa e^{-ik.v} in shared memory, two frequencies per 16-byte word; after a __syncwarp the 32 triangle lanes read
// the A_v of their three corners (one LDS.128 per corner and frequency pair).
//
// Arithmetic of the generic pair.  With nodes x_j = k.v_j, E_j = e^{-i x_j} and gaps
// p = x_1-x_0, q = x_2-x_0, r = q-p, eq. 9 is  g = sum_j c_j E_j  with REAL coefficients
//     c_0 = -1/(pq),  c_1 = 1/(pr),  c_2 = -1/(qr)        (one MUFU.RCP of pqr),
// and its node derivatives (the closed form of PAPER.md:171-173 eq. 11 with reading R2, regrouped) are
//     dg/dx_1 = q (c_0^2 (E_0-E_1) - c_2^2 (E_2-E_1)) - i c_1 E_1
//     dg/dx_2 = p (c_0^2 (E_0-E_1) + (c_1^2-c_0^2) (E_2-E_1)) - i c_2 E_2
//     dg/dx_0 = -i g - dg/dx_1 - dg/dx_2.
// With A_j = kappa E_j the four real numbers a pair contributes are
//     s0 = Re(kappa g),  sI = Im(kappa g),  sb = Re(kappa dg/dx_1),  sc = Re(kappa dg/dx_2),
// all taken on differences of the A_j (every coefficient triple sums to zero).
// Phases advance along z by one complex rotation (rotor e^{-i kstep_z v_z} built in fp64 by the geometry pre-pass) and
// are re-seeded every SEG (8, 16 or 32) frequencies from exact values: the exact phase at the start of a "super-segment"
// of (n_tab+1) SEG frequencies (32-bit integer turns, one accurate sincospi) times a row-independent table of exact
// z-phases kept in shared memory.  Rows longer than one super-segment are walked super-segment by super-segment, so the
// kernel has no limit on N_z.
//
// Near-degenerate pairs (reading R4).  The derivative coefficients grow like 1/(gap^2 gap'), so a pair
// with  m1^2 m2 <= tau_b  (m1 <= m2 the two smallest |gaps|)  is excluded from the fast sums (it accumulates nothing;
// its reciprocal may be inf) and flagged in a per-thread bit mask.  After each chunk of 32 frequencies the lanes' flag
// WORDS are appended, in lane order (one ballot and one 16-byte store per lane), to a ring buffer the WARP keeps in shared
// memory ACROSS chunks and rows; whenever the buffer holds 32 pairs the warp evaluates them, one pair per lane whatever its owner (the series branch
// where all gaps are small, the branch-free far-pair variant otherwise) -- always a full round, the remainder waits for the
// next chunk.  Pair e of a round is found from a prefix sum of the words' bit counts, one warp reduce-or and an n-th-set-bit
// select.  A segmented warp scan sums the results of one (row, owner) run, and the run's last lane hands them to the owner
// lane, which adds them, weighted with the run's k_x, k_y, to its 13 register sums -- lowest lane first (atomicMin on a slot
// table), i.e. in queue order: a fixed order, so the result is bitwise reproducible (reading R22), and the divergent work is
// spread evenly over the lanes.
#pragma once
#include "dm_kernels.cuh"
#include "dm_patches.h"

#define DM_BF_THREADS 32        // one warp = one patch per CTA: the warps share nothing, and a one-warp CTA addresses its
                                // shared memory with constants
#ifndef DM_BF_MINCTA
#define DM_BF_MINCTA 20        // resident CTAs (= warps) per SM the register allocation aims at (<= 102 registers)
#endif
#define DM_BF_CHUNK 32          // frequencies per chunk = one flag word per thread
#ifndef DM_BF_STAGE
#define DM_BF_STAGE 8
#endif                          // frequencies whose vertex phases are staged in shared memory at a time
#define DM_BF_NTAB_MAX 8        // seed-table entries per vertex slot: a super-segment is (n_tab + 1) * SEG frequencies
#define DM_BF_QCAP 64           // ring buffer of flag words per warp: < 32 carried over + <= 32 new per chunk
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
                                  DmGridDev grid, float4* __restrict__ trec, float4* __restrict__ vrec)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= pt.n_lanes) return;
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
        const float ed[3] = {ec[0] - eb[0], ec[1] - eb[1], ec[2] - eb[2]};
        const float a2 = eb[0] * eb[0] + eb[1] * eb[1] + eb[2] * eb[2], b2 = ec[0] * ec[0] + ec[1] * ec[1] + ec[2] * ec[2],
                    c2 = ed[0] * ed[0] + ed[1] * ed[1] + ed[2] * ed[2];
        const float wf = grid.face_w ? grid.face_w[f] : 1.0f;   // density weight of the face
        const float mn = wf * sqrtf(m[0] * m[0] + m[1] * m[1] + m[2] * m[2]);
        m[0] *= wf, m[1] *= wf, m[2] *= wf;
        float4* o = trec + (size_t)DM_BF_TREC * i;
        o[0] = make_float4(__uint_as_float(u[0]), __uint_as_float(u[1]), __uint_as_float(u[2]), __uint_as_float(pt.loc[i]));
        o[1] = make_float4(eb[0], eb[1], eb[2], fmaxf(fmaxf(a2, b2), c2));   // .w: the triangle's longest squared edge
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
}

// ---- kappa pre-pass: everything of the backward that depends on the frequency only ------------------------------------
//   surface: kappa = conj(G);   volume: kappa = i conj(G) / |k|^2  (0 at k = 0: that row is handled by dm_k_corner_grads);
//   zero outside the narrow band (the cotangent there is ignored).  Same layout as G, slab rows only.
template <int MODE>
__global__ void dm_k_kappa(const float2* __restrict__ G, DmGridDev grid, int ix_begin, int ix_end, float2* __restrict__ kappa)
{
    const long long n_slab = (long long)(ix_end - ix_begin) * grid.ny * grid.nzh;
    const long long l = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (l >= n_slab) return;
    const int iz = (int)(l % grid.nzh), iy = (int)((l / grid.nzh) % grid.ny);
    const int ix = ix_begin + (int)(l / ((long long)grid.nzh * grid.ny));
    const int nx = dm_signed_freq(ix, grid.nx), ny = dm_signed_freq(iy, grid.ny);
    const size_t o = ((size_t)ix * grid.ny + iy) * grid.nzh + iz;
    float2 Gk = G[o];
    if (!dm_in_band(grid, nx, ny, iz)) Gk = make_float2(0.f, 0.f);
    float2 out;
    if (MODE == 1) {
        out = make_float2(Gk.x, -Gk.y);
    } else {
        const float kx = grid.kstep[0] * nx, ky = grid.kstep[1] * ny, kz = grid.kstep[2] * iz;
        const float k2 = kx * kx + ky * ky + kz * kz;
        const float inv_k2 = (k2 > 0.f) ? 1.0f / k2 : 0.f;
        out = make_float2(Gk.y * inv_k2, Gk.x * inv_k2);
    }
    kappa[o] = out;
}

// shared memory of one warp = one CTA (static, so every access is base + constant offset)
struct DmBfWarp {
    float4 at4[DM_BF_STAGE / 2][DM_PATCH_MAXV];  // A_v of the patch's vertex slots, two frequencies per word
    float4 rec[32 * DM_BF_TREC];                 // the patch's triangle records (the pooled path reads other lanes')
    uint4 wq[DM_BF_QCAP];                        // ring buffer of flag words: (row_local << 17 | owner << 12 | z of bit 0,
                                                 //   flag word, n_x & 0xffff | n_y << 16, -)
    float2 ztab[DM_BF_NTAB_MAX][32];             // seed table: e^{-2 pi i ((a+1) SEG) u_z} of the lanes' vertex slots
    float2 kbuf[DM_BF_CHUNK];                    // kappa of the chunk's frequencies
    int src[32];                                 // pooled path: the lane that holds the sums of owner l this round
};

// what the pairs of one row add: plain sums and sums weighted with the z index of the frequency
struct DmBfRow {
    float S0, T0, SI, TI, SB, TB, SC, TC;
};

// The fast evaluation of ONE pair (generic closed form) from the staged A_j = kappa e^{-i x_j} of its three corners.
// An excluded (flagged) pair sets `bit` in `flags` instead and accumulates nothing: the seven accumulations and the flag
// are ONE predicated PTX block (the compiler would otherwise merge the two outcomes with a select per sum).
// zf = z index of the frequency; the gaps are p = prow + zf dpz etc. with dpz = kstep_z eb.z (one rounding more than
// k_z eb.z, far below the gaps' own error).
template <int MODE>
__device__ __forceinline__ void dm_bf_pair(const float zf, const float A0r, const float A0i, const float A1r, const float A1i,
                                           const float A2r, const float A2i, const float prow, const float qrow,
                                           const float omrow, const float dpz, const float dqz, const float dmz,
                                           const float tau_k, DmBfRow& rs, uint32_t& flags, const uint32_t bit)
{
    const float p = fmaf(zf, dpz, prow), q = fmaf(zf, dqz, qrow), r = q - p;
    const float pqr = (p * q) * r;
    // the largest derivative coefficient is 1/(m1^2 m2), m1 <= m2 <= m3 the sorted |gaps| (m3 = m1 + m2 always): the pair
    // leaves the fast path when m1^2 m2 = m1 |pqr| / m3 <= tau_k  (also catches p = q = r = 0); tau_k = the threshold of
    // this triangle on this row (tau_b, larger for a triangle that is coarse for the grid)
    const float m1 = fminf(fminf(fabsf(p), fabsf(q)), fabsf(r));
    const float m3 = fmaxf(fmaxf(fabsf(p), fabsf(q)), fabsf(r));
    const float lhs = m1 * fabsf(pqr), rhs = tau_k * m3;     // good = lhs > rhs
    const float R = dm_rcp_approx(pqr);                      // inf / NaN for an excluded pair: never accumulated
    const float c0 = -r * R, c1 = q * R, c2 = -p * R;
    const float c0s = c0 * c0, c1s = c1 * c1, c2s = c2 * c2;
    const float d01r = A0r - A1r, d21r = A2r - A1r;
    const float d01i = A0i - A1i, d21i = A2i - A1i;
    const float s0 = fmaf(c0, d01r, c2 * d21r);
    float sI = fmaf(c0, d01i, c2 * d21i);
    const float t0 = c0s * d01r;
    float sb = fmaf(q, fmaf(-c2s, d21r, t0), c1 * A1i);
    float sc = fmaf(p, fmaf(c1s - c0s, d21r, t0), c2 * A2i);
    if (MODE == 0) {  // volume: omega = k.m_T weights the derivative sums, Q needs k s0
        const float om = fmaf(zf, dmz, omrow);
        sI *= om;
        sb *= om;
        sc *= om;
        asm("{\n\t.reg .pred g;\n\tsetp.gt.f32 g, %9, %10;\n\t"
            "@g add.f32 %0, %0, %11;\n\t@g fma.rn.f32 %1, %15, %11, %1;\n\t"
            "@g add.f32 %2, %2, %12;\n\t@g fma.rn.f32 %3, %15, %12, %3;\n\t"
            "@g add.f32 %4, %4, %13;\n\t@g fma.rn.f32 %5, %15, %13, %5;\n\t"
            "@g add.f32 %6, %6, %14;\n\t@g fma.rn.f32 %7, %15, %14, %7;\n\t"
            "@!g or.b32 %8, %8, %16;\n\t}"
            : "+f"(rs.S0), "+f"(rs.T0), "+f"(rs.SI), "+f"(rs.TI), "+f"(rs.SB), "+f"(rs.TB), "+f"(rs.SC), "+f"(rs.TC), "+r"(flags)
            : "f"(lhs), "f"(rhs), "f"(s0), "f"(sI), "f"(sb), "f"(sc), "f"(zf), "r"(bit));
    } else {
        asm("{\n\t.reg .pred g;\n\tsetp.gt.f32 g, %8, %9;\n\t"
            "@g add.f32 %0, %0, %10;\n\t"
            "@g add.f32 %1, %1, %11;\n\t@g fma.rn.f32 %2, %14, %11, %2;\n\t"
            "@g add.f32 %3, %3, %12;\n\t@g fma.rn.f32 %4, %14, %12, %4;\n\t"
            "@g add.f32 %5, %5, %13;\n\t@g fma.rn.f32 %6, %14, %13, %6;\n\t"
            "@!g or.b32 %7, %7, %15;\n\t}"
            : "+f"(rs.S0), "+f"(rs.SI), "+f"(rs.TI), "+f"(rs.SB), "+f"(rs.TB), "+f"(rs.SC), "+f"(rs.TC), "+r"(flags)
            : "f"(lhs), "f"(rhs), "f"(s0), "f"(sI), "f"(sb), "f"(sc), "f"(zf), "r"(bit));
    }
}

// position of the k-th (0-based) set bit of w (k < popc(w))
__device__ __forceinline__ int dm_nth_set_bit(uint32_t w, int k)
{
    int pos = 0;
#pragma unroll
    for (int h = 16; h > 0; h >>= 1) {
        const int c = __popc(w & ((1u << h) - 1u));
        const bool up = k >= c;
        k -= up ? c : 0;
        pos += up ? h : 0;
        w = up ? (w >> h) : w;
    }
    return pos;
}

// Queue of the pooled slow path (all warp-uniform): wh = ring position of the oldest flag word, wn = flag words queued,
// count = flagged pairs queued, skip = pairs of the oldest word already evaluated.
struct DmBfQueue {
    int wh, wn, count, skip;
};

// One round of the pooled slow path: the n (<= 32) oldest queued pairs of the warp, one per lane whatever its owner.
// Lane l looks at the l-th queued flag word; a prefix sum of the words' bit counts tells lane e which word and which of
// its bits is pair e.  The results of one (row, owner) run are summed by a segmented scan and handed to the owner lane,
// which adds them, weighted with the run's k_x, k_y, to its 13 sums acc[] -- in queue order (reading R22).
// kbase = kappa of (row_begin, z = 0).
template <int MODE>
__device__ __forceinline__ void dm_bf_round(DmBfWarp& W, const int lane, const int n, DmBfQueue& Q, const DmGridDev& grid,
                                            const float2* __restrict__ kbase, float (&acc)[DM_BWD_NSUM])
{
    const uint32_t full = 0xffffffffu;
    uint4 ent = make_uint4(0u, 0u, 0u, 0u);
    if (lane < Q.wn) ent = W.wq[(Q.wh + lane) & (DM_BF_QCAP - 1)];
    const int cnt = __popc(ent.y) - (lane == 0 ? Q.skip : 0);
    int off = cnt;  // inclusive prefix sum of the pairs per word
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int t = __shfl_up_sync(full, off, o);
        if (lane >= o) off += t;
    }
    const bool have = lane < n;
    // the word that holds pair `lane`: every queued word holds at least one pair, so it is the number of words that start
    // at or before the pair, minus one
    const uint32_t starts = __reduce_or_sync(full, (lane < Q.wn && off - cnt < 32) ? (1u << (off - cnt)) : 0u);
    const int src = have ? __popc(starts & (full >> (31 - lane))) - 1 : 0;
    const int s_first = __shfl_sync(full, off - cnt, src);        // index of the word's first unevaluated pair
    const uint32_t s_base = __shfl_sync(full, ent.x, src), s_word = __shfl_sync(full, ent.y, src),
                   s_freq = __shfl_sync(full, ent.z, src);
    const int kbit = have ? lane - s_first + (src == 0 ? Q.skip : 0) : 0;
    const uint32_t code = s_base + (uint32_t)dm_nth_set_bit(s_word, kbit);
    // consume: whole words whose pairs are all in this round; the next word may be evaluated in part
    {
        const int n_done = __popc(__ballot_sync(full, lane < Q.wn && off <= n));
        const int first_nd = __shfl_sync(full, off - cnt, n_done & 31);   // first pair index of the first word not finished
        int skip = 0;
        if (n_done < Q.wn && n_done < 32 && first_nd < n) skip = n - first_nd + (n_done == 0 ? Q.skip : 0);
        Q.wh = (Q.wh + n_done) & (DM_BF_QCAP - 1);
        Q.wn -= n_done;
        Q.count -= n;
        Q.skip = skip;
    }
    const int z = (int)(code & 4095u), own = (int)((code >> 12) & 31u);
    const int rowl = (int)(code >> 17);
    float2 kk = make_float2(0.f, 0.f);                     // (issued early: an L2 access)
    if (have) kk = kbase[(size_t)rowl * grid.nzh + z];
    const int nx = (int)(short)(s_freq & 0xffffu), ny = (int)(short)(s_freq >> 16);
    const float kx = grid.kstep[0] * nx, ky = grid.kstep[1] * ny, kz = grid.kstep[2] * (float)z;
    const float4* orc = W.rec + own * DM_BF_TREC;
    const float4 q0 = orc[0], q3 = orc[1], q4 = orc[2];
    const float p = fmaf(kz, q3.z, fmaf(kx, q3.x, ky * q3.y));
    const float q = fmaf(kz, q4.z, fmaf(kx, q4.x, ky * q4.y));
    const bool series = fmaxf(fmaxf(fabsf(p), fabsf(q)), fabsf(q - p)) < DM_SERIES_RADIUS;
    cf psi = {0.f, 0.f}, dp = {0.f, 0.f}, dq = {0.f, 0.f};
    if (__any_sync(full, have && series)) {
        cf a, b, c;
        dm_psi_series<true>(series ? p : 0.f, series ? q : 0.f, a, b, c);
        if (series) { psi = a; dp = b; dq = c; }
    }
    if (__any_sync(full, have && !series)) {
        cf a, b, c;
        dm_psi_far_uniform(series ? 0.f : p, series ? 1.f : q, a, b, c);
        if (!series) { psi = a; dp = b; dq = c; }
    }
    const cf E = dm_expmi_turns_fast(dm_phase_turns(nx, ny, z, __float_as_uint(q0.x), __float_as_uint(q0.y),
                                                    __float_as_uint(q0.z)));
    const cf kE = cmul(cf{kk.x, kk.y}, E);
    const cf kg = cmul(kE, psi);
    // v[0..3] = s0, sI, sb, sc (the last three weighted with omega in volume mode), v[4..7] = k_z times them
    float v[8];
    v[0] = kg.re;
    v[1] = kg.im;
    v[2] = kE.re * dp.re - kE.im * dp.im;
    v[3] = kE.re * dq.re - kE.im * dq.im;
    if (MODE == 0) {
        const float4 q5 = orc[3];
        const float om = fmaf(kz, q5.z, fmaf(kx, q5.x, ky * q5.y));
        v[1] *= om;
        v[2] *= om;
        v[3] *= om;
    }
#pragma unroll
    for (int i = 0; i < 4; ++i) v[4 + i] = kz * v[i];
    // segmented inclusive scan over the runs of equal (row, owner): head flags from adjacent keys
    const uint32_t key = have ? (code >> 12) : (0xffffff00u | (uint32_t)lane);
    const uint32_t kprev = __shfl_up_sync(full, key, 1);
    const uint32_t heads = __ballot_sync(full, lane == 0 || kprev != key);
    const int dist = lane - (31 - __clz((int)(heads & (full >> (31 - lane)))));   // distance to the run's first lane
    const int maxdist = __reduce_max_sync(full, dist);
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        if (o <= maxdist) {   // warp-uniform: most rounds hold short runs only
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                if (MODE == 1 && i == 4) continue;  // k_z s0 is a volume-mode sum
                const float x = __shfl_up_sync(full, v[i], o);
                if (o <= dist) v[i] += x;
            }
        }
    }
    // hand every run's sums to its owner lane.  Two runs of one owner (different rows or chunks) can end in the same
    // round: the lowest lane goes first (atomicMin), the others in later passes -- queue order.
    bool pending = have && (lane == 31 || ((heads >> (lane + 1)) & 1u));
    do {
        W.src[lane] = 255;
        __syncwarp();
        if (pending) atomicMin(&W.src[own], lane);
        __syncwarp();
        const int s = W.src[lane];
        if (pending && W.src[own] == lane) pending = false;
        const bool got = s < 32;
        const int sl = got ? s : 0;
        const float gkx = __shfl_sync(full, kx, sl), gky = __shfl_sync(full, ky, sl);
        float g[8];
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            if (MODE == 1 && i == 4) continue;
            g[i] = __shfl_sync(full, v[i], sl);
        }
        if (got) {
            if (MODE == 1) {
                acc[0] += g[0];
            } else {
                acc[1] = fmaf(gkx, g[0], acc[1]);
                acc[2] = fmaf(gky, g[0], acc[2]);
                acc[3] += g[4];
            }
#pragma unroll
            for (int i = 1; i < 4; ++i) {
                acc[1 + 3 * i] = fmaf(gkx, g[i], acc[1 + 3 * i]);
                acc[2 + 3 * i] = fmaf(gky, g[i], acc[2 + 3 * i]);
                acc[3 + 3 * i] += g[4 + i];
            }
        }
        __syncwarp();
    } while (__any_sync(full, pending));
}

// ---- A6 backward, fast kernel -----------------------------------------------------------------------------------
// grid = (n_patches, n_split), one warp per CTA = one patch; part[(split*13 + s)*n_faces + face] as in
// dm_k_backward_robust.  BAND = the narrow band is set (band_z holds the in-band z interval of every row).
// SEG = frequencies between exact phase seeds (8, 16 or 32), n_tab <= DM_BF_NTAB_MAX the seed-table entries per vertex
// slot (a super-segment is (n_tab + 1) SEG frequencies); both chosen by the host.  rows_per_split <= 32768.
template <int MODE, int SEG, bool BAND>
__global__ void __launch_bounds__(32, DM_BF_MINCTA)
dm_k_backward_fast(const float4* __restrict__ trec_g, const float4* __restrict__ vrec_g, DmPatchDev pt, int n_faces,
                   DmGridDev grid, int ix_begin, int ix_end, int rows_per_split, float tau_b, int n_tab,
                   const float2* __restrict__ kappa, const int2* __restrict__ band_z, float* __restrict__ part)
{
    static_assert(SEG == 8 || SEG == 16 || SEG == 32, "SEG is a multiple of the stage and divides the chunk");
    __shared__ DmBfWarp W;
    const int lane = threadIdx.x;
    const int gl = blockIdx.x * 32 + lane;                 // global lane = 32 * patch + lane
    const int face = pt.face[gl];
    const bool live = face >= 0;
    float dpz, dqz, dmz;
    const float4 *pa0, *pa1, *pa2;                         // the staged phases of the triangle's corners
    {
        const float4 r0 = trec_g[(size_t)DM_BF_TREC * gl], r1 = trec_g[(size_t)DM_BF_TREC * gl + 1],
                     r2 = trec_g[(size_t)DM_BF_TREC * gl + 2], r3 = trec_g[(size_t)DM_BF_TREC * gl + 3];
        W.rec[lane * DM_BF_TREC + 0] = r0;
        W.rec[lane * DM_BF_TREC + 1] = r1;
        W.rec[lane * DM_BF_TREC + 2] = r2;
        W.rec[lane * DM_BF_TREC + 3] = r3;
        const uint32_t loc = __float_as_uint(r0.w);
        pa0 = &W.at4[0][loc & 255u], pa1 = &W.at4[0][(loc >> 8) & 255u], pa2 = &W.at4[0][(loc >> 16) & 255u];
        dpz = grid.kstep[2] * r1.z, dqz = grid.kstep[2] * r2.z, dmz = grid.kstep[2] * r3.z;
    }
    // the vertex slot this lane owns (slot lane of its patch)
    const float4 va0 = vrec_g[(size_t)DM_BF_VREC * gl], va1 = vrec_g[(size_t)DM_BF_VREC * gl + 1];
    const uint32_t uax = __float_as_uint(va0.x), uay = __float_as_uint(va0.y), uaz = __float_as_uint(va0.z);
    const cf rhoa = {va0.w, va1.x};
    const int nzh = grid.nzh;
    const int n_rows = (ix_end - ix_begin) * grid.ny;
    const int row_begin = blockIdx.y * rows_per_split;
    const int row_end = min(n_rows, row_begin + rows_per_split);
    const int SS = (n_tab + 1) * SEG;                      // frequencies per super-segment

    // seed table (row-independent): exact z-phases of this lane's vertex slot at the multiples of SEG
    for (int a = 0; a < n_tab; ++a) {
        const cf z0 = dm_expmi_turns((uint32_t)((a + 1) * SEG) * uaz);
        W.ztab[a][lane] = make_float2(z0.re, z0.im);
    }
    __syncwarp();

    // acc: [0] S0 | [1..3] Q | [4..6] W | [7..9] Vb | [10..12] Vc   (dm_k_backward_robust)
    float acc[DM_BWD_NSUM];
#pragma unroll
    for (int s = 0; s < DM_BWD_NSUM; ++s) acc[s] = 0.f;
    DmBfQueue Q = {0, 0, 0, 0};                            // flag words waiting for the pooled path (warp-uniform)

    // in-band z interval of a row, started at a seed position (the whole row without a band)
    auto row_range = [&](int row, int& lo, int& hi) {
        lo = 0, hi = nzh;
        if (BAND) {
            const int2 bz = band_z[ix_begin * grid.ny + row];
            lo = bz.x & ~(SEG - 1);
            hi = bz.y;
        }
    };
    const float2* const kbase = kappa + ((size_t)ix_begin * grid.ny + row_begin) * nzh;
    const float2* krow = kbase;
    float2 knext = make_float2(0.f, 0.f);                  // kappa of this lane's frequency of the NEXT chunk
    int pref_row = -1;                                     // row whose first chunk knext holds
    int ix = ix_begin + row_begin / grid.ny, iy = row_begin % grid.ny;

    for (int row = row_begin; row < row_end; ++row, krow += nzh) {
        int z_lo, z_hi;
        row_range(row, z_lo, z_hi);
        int zn_lo = 0, zn_hi = 0;                          // the next row's interval (for the prefetch)
        if (row + 1 < row_end) row_range(row + 1, zn_lo, zn_hi);
        const int nx = dm_signed_freq(ix, grid.nx), ny = dm_signed_freq(iy, grid.ny);
        if (++iy == grid.ny) iy = 0, ++ix;
        if (z_lo >= z_hi) continue;
        const int rowl = row - row_begin;
        const float kx = grid.kstep[0] * nx, ky = grid.kstep[1] * ny;
        float prow, qrow, omrow, tau_row;
        {
            const float4 r1 = W.rec[lane * DM_BF_TREC + 1], r2 = W.rec[lane * DM_BF_TREC + 2], r3 = W.rec[lane * DM_BF_TREC + 3];
            prow = fmaf(kx, r1.x, ky * r1.y), qrow = fmaf(kx, r2.x, ky * r2.y), omrow = fmaf(kx, r3.x, ky * r3.y);
            // flag threshold of this triangle on this row: tau_b max(1, (|k| h_T / 12)^3), |k| the largest of the row, h_T
            // the longest edge of the triangle.  On a triangle that is large for the grid (|k| h >> 1) the rounding error of
            // a gap k.e grows like |k| h while the integral decays like 1/(|k| h)^2; the factor is 1 when |k| h_T <= 12
            const float kzm = grid.kstep[2] * (float)(nzh - 1);
            const float kh2 = (1.0f / 144.0f) * (kx * kx + ky * ky + kzm * kzm) * r1.w;
            tau_row = tau_b * fmaxf(1.0f, kh2 * sqrtf(kh2));
        }
        const uint32_t xturns = (uint32_t)nx * uax + (uint32_t)ny * uay;   // exact row phase of the lane's vertex slot
        if (pref_row != row) knext = (z_lo + lane < z_hi) ? krow[z_lo + lane] : make_float2(0.f, 0.f);
        DmBfRow rs = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
        cf Xs = {1.f, 0.f}, Ea = {1.f, 0.f};
        int zs = z_lo, ze = z_lo;                          // current super-segment [zs, ze)
        const float2* ztp = &W.ztab[0][lane];              // next seed-table entry of the super-segment
        for (int z = z_lo; z < z_hi;) {
            if (z == ze) {                                 // a new super-segment: exact phase at its start
                zs = z;
                ze = min(zs + SS, z_hi);
                Xs = dm_expmi_turns(xturns + (uint32_t)zs * uaz);
                Ea = Xs;
                ztp = &W.ztab[0][lane];
            }
            const int clen = min(DM_BF_CHUNK, ze - z);
            // ---- stage kappa of the chunk, prefetch the next chunk's (entries past its end are loaded, never read) ----
            W.kbuf[lane] = knext;
            __syncwarp();
            {
                const int zn = z + clen;
                if (zn < z_hi) {
                    knext = (zn + lane < z_hi) ? krow[zn + lane] : make_float2(0.f, 0.f);
                } else if (zn_lo < zn_hi) {
                    knext = (zn_lo + lane < zn_hi) ? krow[nzh + zn_lo + lane] : make_float2(0.f, 0.f);
                    pref_row = row + 1;
                }
            }
            // ---- fast pass over the chunk: bodies of DM_BF_STAGE frequencies, exact seeds every SEG -----------------
            uint32_t word = 0;
            float zf = (float)z;
            const float4* kb4 = reinterpret_cast<const float4*>(W.kbuf);
            int zloc = 0;
#pragma unroll 1
            for (; zloc + DM_BF_STAGE <= clen; zloc += DM_BF_STAGE, zf += (float)DM_BF_STAGE, kb4 += DM_BF_STAGE / 2) {
                if ((SEG <= DM_BF_STAGE || ((z + zloc - zs) & (SEG - 1)) == 0) && z + zloc != zs) {   // exact seed
                    const float2 a0 = *ztp;
                    ztp += 32;
                    Ea = cmul(Xs, cf{a0.x, a0.y});
                }
                // every lane writes A_v of its vertex slot for 8 frequencies, then evaluates its triangle at them
#pragma unroll
                for (int jp = 0; jp < DM_BF_STAGE / 2; ++jp) {
                    if (SEG < DM_BF_STAGE && jp > 0 && (2 * jp) % SEG == 0) {   // a seed inside the body
                        const float2 a0 = *ztp;
                        ztp += 32;
                        Ea = cmul(Xs, cf{a0.x, a0.y});
                    }
                    const float4 k4 = kb4[jp];
                    const cf A = cmul(cf{k4.x, k4.y}, Ea);
                    Ea = cmul(Ea, rhoa);
                    const cf B = cmul(cf{k4.z, k4.w}, Ea);
                    Ea = cmul(Ea, rhoa);
                    W.at4[jp][lane] = make_float4(A.re, A.im, B.re, B.im);
                }
                __syncwarp();
                uint32_t sf = 0;
#pragma unroll
                for (int jp = 0; jp < DM_BF_STAGE / 2; ++jp) {
                    const float4 a0 = pa0[jp * DM_PATCH_MAXV], a1 = pa1[jp * DM_PATCH_MAXV], a2 = pa2[jp * DM_PATCH_MAXV];
                    dm_bf_pair<MODE>(zf + (float)(2 * jp), a0.x, a0.y, a1.x, a1.y, a2.x, a2.y, prow, qrow, omrow, dpz, dqz, dmz,
                                     tau_row, rs, sf, 1u << (2 * jp));
                    dm_bf_pair<MODE>(zf + (float)(2 * jp + 1), a0.z, a0.w, a1.z, a1.w, a2.z, a2.w, prow, qrow, omrow, dpz, dqz,
                                     dmz, tau_row, rs, sf, 1u << (2 * jp + 1));
                }
                __syncwarp();
                word |= sf << zloc;
            }
            if (zloc < clen) {
                // ragged end of the chunk: one frequency at a time
#pragma unroll 1
                for (; zloc < clen; ++zloc, zf += 1.0f) {
                    if (((z + zloc - zs) & (SEG - 1)) == 0 && z + zloc != zs) {   // exact seed
                        const float2 a0 = *ztp;
                        ztp += 32;
                        Ea = cmul(Xs, cf{a0.x, a0.y});
                    }
                    const float2 k1 = W.kbuf[zloc];
                    const cf A = cmul(cf{k1.x, k1.y}, Ea);
                    Ea = cmul(Ea, rhoa);
                    W.at4[0][lane] = make_float4(A.re, A.im, 0.f, 0.f);
                    __syncwarp();
                    const float4 a0 = pa0[0], a1 = pa1[0], a2 = pa2[0];
                    dm_bf_pair<MODE>(zf, a0.x, a0.y, a1.x, a1.y, a2.x, a2.y, prow, qrow, omrow, dpz, dqz, dmz, tau_row, rs, word,
                                     1u << zloc);
                    __syncwarp();
                }
            }
            word = live ? word : 0u;
            // ---- queue the chunk's flag words in lane order; evaluate whole rounds of 32 pairs ------------------------
            {
                const uint32_t m = __ballot_sync(0xffffffffu, word != 0u);
                if (m != 0u) {
                    if (word != 0u)
                        W.wq[(Q.wh + Q.wn + __popc(m & ((1u << lane) - 1u))) & (DM_BF_QCAP - 1)] =
                            make_uint4(((uint32_t)rowl << 17) | ((uint32_t)lane << 12) | (uint32_t)z, word,
                                       ((uint32_t)nx & 0xffffu) | ((uint32_t)ny << 16), 0u);
                    Q.wn += __popc(m);
                    Q.count += __reduce_add_sync(0xffffffffu, __popc(word));
                    __syncwarp();
                    while (Q.count >= 32) dm_bf_round<MODE>(W, lane, 32, Q, grid, kbase, acc);
                }
            }
            z += clen;
        }
        // fold the row into the 13 sums (the z-weighted sums carry the z index: k_z = kstep_z z)
        if (MODE == 1) {
            acc[0] += rs.S0;
        } else {
            acc[1] = fmaf(kx, rs.S0, acc[1]);
            acc[2] = fmaf(ky, rs.S0, acc[2]);
            acc[3] = fmaf(grid.kstep[2], rs.T0, acc[3]);
        }
        acc[4] = fmaf(kx, rs.SI, acc[4]);
        acc[5] = fmaf(ky, rs.SI, acc[5]);
        acc[6] = fmaf(grid.kstep[2], rs.TI, acc[6]);
        acc[7] = fmaf(kx, rs.SB, acc[7]);
        acc[8] = fmaf(ky, rs.SB, acc[8]);
        acc[9] = fmaf(grid.kstep[2], rs.TB, acc[9]);
        acc[10] = fmaf(kx, rs.SC, acc[10]);
        acc[11] = fmaf(ky, rs.SC, acc[11]);
        acc[12] = fmaf(grid.kstep[2], rs.TC, acc[12]);
    }
    if (Q.count > 0) dm_bf_round<MODE>(W, lane, Q.count, Q, grid, kbase, acc);   // the pairs still queued (< 32)
    if (live) {
#pragma unroll
        for (int s = 0; s < DM_BWD_NSUM; ++s) part[((size_t)blockIdx.y * DM_BWD_NSUM + s) * n_faces + face] = acc[s];
    }
}
