// deltamic.cu -- plan object and C ABI (include/deltamic.h) of the B200-native deltaMic mesh Fourier transform.
// Host logic only; the arithmetic lives in dm_math.cuh / dm_kernels.cuh / dm_fast.cuh.
#include <cuda_runtime.h>
#include <cufft.h>

#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <utility>
#include <vector>

#include "../../include/deltamic.h"
#include "dm_fast.cuh"
#include "dm_bwd_fast.cuh"
#include "dm_strips.h"
#include "dm_splits.h"
#include "dm_shape.cuh"

#define DM_VERSION 100
#ifndef DM_BWD_SPLIT_TARGET
#define DM_BWD_SPLIT_TARGET 192  // k-splits of the backward: (128-triangle blocks x splits) per SM
#endif

struct dm_plan {
    dm_grid grid;
    DmGridDev gd;
    int mode;
    int32_t n_vertices, n_faces;
    int ix_begin, ix_end;
    cudaStream_t stream;
    int n_sm;
    // device workspace
    int32_t* faces = nullptr;        // [n_faces*3]
    int32_t* csr_off = nullptr;      // [n_vertices+1]
    int32_t* csr_corner = nullptr;   // [n_faces*3]   3*face+corner, ascending per vertex
    float4* rec = nullptr;           // [n_faces*4]   triangle records (A1)
    // patches of the fast backward kernel (topology only; built at create) and its per-call records
    int32_t *pt_face = nullptr, *pt_vid = nullptr;
    uint32_t* pt_loc = nullptr;
    int pt_lanes = 0;                // 32 * patches, padded to a multiple of DM_BF_THREADS
    float4* btrec = nullptr;         // [pt_lanes*DM_BF_TREC] backward triangle records (A1)
    float4* bvrec = nullptr;         // [pt_lanes*DM_BF_VREC] backward vertex-slot records (A1)
    float* part = nullptr;           // [n_split_max*13*n_faces]
    float* corner = nullptr;         // [n_faces*9]
    float2* spec = nullptr;          // [n_k] scratch spectrum (S, R or G)
    float2* spec2 = nullptr;         // [n_k] G inside dm_render_backward
    int n_split_max = 0;
    // strip walk of the fast forward kernel (topology only; built at create)
    int32_t *st_new = nullptr, *st_prev = nullptr, *st_ret = nullptr, *st_fid = nullptr, *st_chunk_off = nullptr;
    int st_n_rec = 0, st_n_chunks = 0;
    float4* st_rec = nullptr;        // [st_n_rec*3] strip records (A1)
    float2* fwd_part = nullptr;      // [st_n_chunks * n_k] per-chunk partial spectra
    unsigned int* hmax2 = nullptr;   // 16 bytes of edge statistics (dm_edge_stats_add), rebuilt every call
    double* dc_part = nullptr;       // [DM_DC_BLOCKS] block sums of the k = 0 entry
    bool normalise = false;          // DM_OPT_AREA_NORMALISED (surface mode): u = F/|Lambda|, eq. 12-13
    double* dc_total = nullptr;      // [1] fp64 volume / total area of the last forward (k = 0 kernels)
    double* dot_part = nullptr;      // [DM_DOT_BLOCKS + 1] block sums and result of sum_k Re(conj(G) F)
    float* face_w = nullptr;         // [n_faces] per-face density weights, valid while gd.face_w points at it
    bool weights_robust = false;     // the weights are outside the regime the fast kernels are validated for (mixed
                                     // sign, or varying inside a connected component in volume mode): every pair goes
                                     // through the robust kernels
    std::vector<int32_t> faces_host; // host copy of the faces (the shape-optimisation state builds the vertex graph from it)
    std::vector<int32_t> face_comp;  // host: connected component (shared vertices) of every face, built at create
    int last_fwd_path = -1, last_bwd_path = -1;   // 0 = fast, 1 = robust: what the last mesh-FT calls actually ran
    long long band_count = 0;        // stored frequencies inside the narrow band (whole grid)
    uint32_t* band_slots = nullptr;  // the forward kernel's thread list under the narrow band
    int2* band_z = nullptr;          // [nx*ny] in-band z interval of every row (narrow band), valid while band_on
    bool band_on = false;
    float2* kappa = nullptr;         // [n_k] kappa(k) of the fast backward kernel (dm_k_kappa), allocated on first use
    float2* spec3 = nullptr;         // [n_k] the forward spectrum F of dm_render (kept for dm_render_backward), or the one
                                     // recomputed for the PSF gradient / eq. 13 (allocated on first use)
    bool F_valid = false;            // spec3 and dc_total belong to the last dm_render and nothing changed them since
    bool reuse_F = false;            // DM_OPT_REUSE_SPECTRUM
    double* psfg_part = nullptr;     // [DM_PSFG_BLOCKS*6] block sums of the PSF gradient
    float* psfg_out = nullptr;       // [6] device result of the PSF gradient
    int fwd_path = 0, bwd_path = 0;  // 0 = fast, 1 = robust
    float tau = 1e-2f, tau_b = 1.2e-4f;
    cufftHandle fft_xy = 0, fft_z = 0, fft_r2c = 0;
    bool have_xy = false, have_z = false, have_r2c = false, have_fft = false;
    // stage timing
    cudaEvent_t ev[8];
    bool ev_ok = false;
    bool stage_ran[4] = {false, false, false, false};
    int64_t launches = 0;
};

namespace {

const char* kErr[] = {"ok", "invalid argument", "bad mesh (face index out of range)", "allocation failed",
                      "CUDA error", "cuFFT error", "unsupported",
                      "mesh too large for the fixed scratch of dm_mesh_ft_forward_noalloc"};

inline size_t n_k_of(const dm_plan* p) { return (size_t)p->gd.nx * p->gd.ny * p->gd.nzh; }

#define DM_CUDA(x)                            \
    do {                                      \
        if ((x) != cudaSuccess) return DM_ERR_CUDA; \
    } while (0)

int check_launch(dm_plan* p, int n = 1)
{
    p->launches += n;
    return cudaGetLastError() == cudaSuccess ? DM_OK : DM_ERR_CUDA;
}

void stage_begin(dm_plan* p, int s)
{
    cudaEventRecord(p->ev[2 * s], p->stream);
}
void stage_end(dm_plan* p, int s)
{
    cudaEventRecord(p->ev[2 * s + 1], p->stream);
    p->stage_ran[s] = true;
}
void stage_reset(dm_plan* p)
{
    for (int s = 0; s < 4; ++s) p->stage_ran[s] = false;
}

int backward_splits(const dm_plan* p, int* rows_per_split)
{
    return dm_backward_splits((p->ix_end - p->ix_begin) * p->gd.ny, p->gd.nzh, p->n_faces, p->n_sm, DM_BWD_SPLIT_TARGET,
                              p->band_on, p->n_split_max, rows_per_split);
}

int make_psf(const dm_plan* p, const float* cov, DmPsfDev* out)
{
    if (!cov) return DM_ERR_INVALID_ARG;
    for (int i = 0; i < 6; ++i) {
        if (!std::isfinite(cov[i])) return DM_ERR_INVALID_ARG;
        out->cov[i] = cov[i];
    }
    for (int d = 0; d < 3; ++d)
        out->org_turns[d] = (double)p->grid.origin[d] / ((double)p->grid.n[d] * (double)p->grid.spacing[d]);
    out->inv_voxel = (float)(1.0 / ((double)p->grid.spacing[0] * p->grid.spacing[1] * p->grid.spacing[2] *
                                    (double)p->grid.n[0] * p->grid.n[1] * p->grid.n[2]));
    return DM_OK;
}

int ensure_fft(dm_plan* p)
{
    if (p->have_fft) return DM_OK;
    const int nx = p->gd.nx, ny = p->gd.ny, nz = p->gd.nz, nzh = p->gd.nzh;
    // inverse = 2D C2C over (x,y) for every stored n_z, then 1D C2R along z  (same order as numpy irfftn, R13)
    int n2[2] = {nx, ny};
    int emb2[2] = {nx, ny};
    if (!p->have_xy) {
        if (cufftPlanMany(&p->fft_xy, 2, n2, emb2, nzh, 1, emb2, nzh, 1, CUFFT_C2C, nzh) != CUFFT_SUCCESS) return DM_ERR_CUFFT;
        p->have_xy = true;
    }
    int n1[1] = {nz};
    int iemb[1] = {nzh}, oemb[1] = {nz};
    if (!p->have_z) {
        if (cufftPlanMany(&p->fft_z, 1, n1, iemb, 1, nzh, oemb, 1, nz, CUFFT_C2R, nx * ny) != CUFFT_SUCCESS) return DM_ERR_CUFFT;
        p->have_z = true;
    }
    if (!p->have_r2c) {
        if (cufftPlan3d(&p->fft_r2c, nx, ny, nz, CUFFT_R2C) != CUFFT_SUCCESS) return DM_ERR_CUFFT;
        p->have_r2c = true;
    }
    if (cufftSetStream(p->fft_xy, p->stream) != CUFFT_SUCCESS || cufftSetStream(p->fft_z, p->stream) != CUFFT_SUCCESS ||
        cufftSetStream(p->fft_r2c, p->stream) != CUFFT_SUCCESS)
        return DM_ERR_CUFFT;
    if (!p->spec2 && cudaMalloc(&p->spec2, n_k_of(p) * sizeof(float2)) != cudaSuccess) return DM_ERR_ALLOC;
    p->have_fft = true;
    return DM_OK;
}

int run_geometry(dm_plan* p, const float* vertices_dev)
{
    dm_k_geometry<<<(p->n_faces + 127) / 128, 128, 0, p->stream>>>(vertices_dev, p->faces, p->n_faces, p->gd, p->rec);
    return check_launch(p);
}

int run_forward_robust(dm_plan* p, const float* vertices_dev, float* F_dev)
{
    int rc = run_geometry(p, vertices_dev);
    if (rc) return rc;
    const long long n_slab = (long long)(p->ix_end - p->ix_begin) * p->gd.ny * p->gd.nzh;
    const unsigned blocks = (unsigned)((n_slab + 127) / 128);
    dm_k_forward_robust<<<blocks, 128, 0, p->stream>>>(p->rec, p->n_faces, p->gd, p->mode, p->ix_begin, p->ix_end,
                                                       (float2*)F_dev);
    return check_launch(p);
}

int run_forward_fast(dm_plan* p, const float* vertices_dev, float* F_dev)
{
    if (cudaMemsetAsync(p->hmax2, 0, 16, p->stream) != cudaSuccess) return DM_ERR_CUDA;
    DmStripDev st = {p->st_new, p->st_prev, p->st_ret, p->st_fid, p->st_n_rec};
    dm_k_strip_geometry<<<(p->st_n_rec + 127) / 128, 128, 0, p->stream>>>(vertices_dev, p->faces, st, p->gd, p->mode,
                                                                           p->st_rec, p->hmax2);
    int rc = check_launch(p);
    if (rc) return rc;
    const int n_yruns = (p->gd.ny + DM_K - 1) / DM_K;
    const long long n_thr = p->gd.band_slots ? (long long)p->gd.n_band_slots
                                             : (long long)(p->ix_end - p->ix_begin) * n_yruns * p->gd.nzh;
    dim3 grid((unsigned)((n_thr + DM_FAST_THREADS - 1) / DM_FAST_THREADS), (unsigned)p->st_n_chunks);
    const size_t stride = n_k_of(p);
    if (p->mode == DM_SURFACE)
        dm_k_forward_fast<1><<<grid, DM_FAST_THREADS, 0, p->stream>>>(p->st_rec, p->st_chunk_off, p->gd, p->ix_begin, p->ix_end,
                                                                      n_yruns, p->tau, p->hmax2, stride, p->fwd_part);
    else
        dm_k_forward_fast<0><<<grid, DM_FAST_THREADS, 0, p->stream>>>(p->st_rec, p->st_chunk_off, p->gd, p->ix_begin, p->ix_end,
                                                                      n_yruns, p->tau, p->hmax2, stride, p->fwd_part);
    if ((rc = check_launch(p))) return rc;
    // candidates of the low-k kernel: the part of its box that exists on this grid, one per thread; only the low ones
    // (|k| h_max < DM_LOWK_RADIUS, decided on the device) cost anything
    const int bx = std::min(DM_LOWK_BOX, p->gd.nx / 2), by = std::min(DM_LOWK_BOX, p->gd.ny / 2), bz = std::min(DM_LOWK_BOX, p->gd.nz / 2);
    const long long n_cand = (long long)(2 * bx + 1) * (2 * by + 1) * (bz + 1);
    const unsigned lowk_blocks = (unsigned)((n_cand + DM_LOWK_CAND - 1) / DM_LOWK_CAND);
    if (p->mode == DM_SURFACE)
        dm_k_forward_lowk<1><<<lowk_blocks, DM_LOWK_THREADS, 0, p->stream>>>(p->st_rec, p->st_chunk_off, p->st_n_chunks, p->gd, p->ix_begin,
                                                                 p->ix_end, bx, by, bz, p->hmax2, (float2*)F_dev);
    else
        dm_k_forward_lowk<0><<<lowk_blocks, DM_LOWK_THREADS, 0, p->stream>>>(p->st_rec, p->st_chunk_off, p->st_n_chunks, p->gd, p->ix_begin,
                                                                 p->ix_end, bx, by, bz, p->hmax2, (float2*)F_dev);
    if ((rc = check_launch(p))) return rc;
    const long long n_slab = (long long)(p->ix_end - p->ix_begin) * p->gd.ny * p->gd.nzh;
    dm_k_forward_finish<<<(unsigned)((n_slab + 255) / 256), 256, 0, p->stream>>>(p->fwd_part, stride, p->st_n_chunks, p->gd,
                                                                                p->ix_begin, p->ix_end, p->hmax2, (float2*)F_dev);
    return check_launch(p);
}

int run_forward_raw(dm_plan* p, const float* vertices_dev, float* F_dev)
{
    const bool robust = p->fwd_path != 0 || p->weights_robust;
    p->last_fwd_path = robust ? 1 : 0;
    int rc = robust ? run_forward_robust(p, vertices_dev, F_dev) : run_forward_fast(p, vertices_dev, F_dev);
    if (rc) return rc;
    if (p->ix_begin == 0) {
        dm_k_dc_partial<<<DM_DC_BLOCKS, 256, 0, p->stream>>>(vertices_dev, p->faces, p->n_faces, p->mode, p->gd.face_w, p->dc_part);
        if ((rc = check_launch(p))) return rc;
        dm_k_dc_final<<<1, DM_DC_BLOCKS, 0, p->stream>>>(p->dc_part, F_dev, p->dc_total);
        rc = check_launch(p);
    }
    return rc;
}

// forward as the caller sees it: the raw mesh FT, divided by the total area in the area-normalised mode (eq. 12)
int run_forward(dm_plan* p, const float* vertices_dev, float* F_dev)
{
    if (p->normalise && (p->ix_begin != 0 || p->ix_end != p->gd.nx)) return DM_ERR_UNSUPPORTED;
    int rc = run_forward_raw(p, vertices_dev, F_dev);
    if (rc || !p->normalise) return rc;
    const long long nk = (long long)n_k_of(p);
    dm_k_scale_spectrum<<<(unsigned)((nk + 255) / 256), 256, 0, p->stream>>>((float2*)F_dev, nk, p->dc_total);
    return check_launch(p);
}

// F_reuse: the (area-normalised) forward spectrum of these vertices when the caller already has it and dc_total still
// holds their total area; nullptr = recompute what eq. 13 needs
int run_backward(dm_plan* p, const float* vertices_dev, const float* G_dev, float* dv_dev, const float2* F_reuse = nullptr)
{
    if (p->normalise && (p->ix_begin != 0 || p->ix_end != p->gd.nx)) return DM_ERR_UNSUPPORTED;   // before any launch
    int rps = 1;
    const int n_split = backward_splits(p, &rps);
    dim3 grid((p->n_faces + 127) / 128, n_split);
    const int nzh = p->gd.nzh;
    // The flag threshold is calibrated for sums over many frequencies (errors of single pairs average out); when a vertex
    // gradient sums fewer than ~5e4 frequencies (tiny grids, narrow bands, thin slabs) one pair just above the threshold
    // could dominate, so the threshold grows like 1/sqrt(number of frequencies)
    // (counted over the whole grid, not the slab: the slabs' partial gradients are summed afterwards)
    double n_freq = (double)p->gd.nx * p->gd.ny * nzh;
    if (p->band_on) n_freq = std::max(1.0, (double)p->band_count);
    const float tau_b_eff = (float)((double)p->tau_b * std::max(1.0, std::sqrt(5.0e4 / n_freq)));
    // seed spacing of the fast kernel (frequencies between exact phase seeds) and the seed-table entries per vertex slot;
    // a row longer than (n_tab + 1) seg frequencies is walked in several super-segments
    const int seg = nzh <= 72 ? 8 : (nzh <= 144 ? 16 : 32);
    const int n_tab = std::min(DM_BF_NTAB_MAX, (nzh + seg - 1) / seg - 1);
    int rc;
    const bool robust = p->bwd_path != 0 || p->weights_robust || rps > DM_SPLIT_MAX_ROWS;
    p->last_bwd_path = robust ? 1 : 0;
    if (!robust) {
        const DmPatchDev pt = {p->pt_face, p->pt_vid, p->pt_loc, p->pt_lanes};
        grid.x = (unsigned)(p->pt_lanes / DM_BF_THREADS);
        const size_t nk = n_k_of(p);
        if (!p->kappa && cudaMalloc(&p->kappa, nk * sizeof(float2)) != cudaSuccess) return DM_ERR_ALLOC;
        dm_k_bwd_geometry<<<(p->pt_lanes + 127) / 128, 128, 0, p->stream>>>(vertices_dev, p->faces, pt, p->gd, p->btrec, p->bvrec);
        if ((rc = check_launch(p))) return rc;
        const long long n_slab = (long long)(p->ix_end - p->ix_begin) * p->gd.ny * nzh;
        if (p->mode == DM_SURFACE)
            dm_k_kappa<1><<<(unsigned)((n_slab + 255) / 256), 256, 0, p->stream>>>((const float2*)G_dev, p->gd, p->ix_begin, p->ix_end, p->kappa);
        else
            dm_k_kappa<0><<<(unsigned)((n_slab + 255) / 256), 256, 0, p->stream>>>((const float2*)G_dev, p->gd, p->ix_begin, p->ix_end, p->kappa);
        if ((rc = check_launch(p))) return rc;
#define DM_LAUNCH_BF2(MODE, SEG, BAND)                                                                                   \
    dm_k_backward_fast<MODE, SEG, BAND><<<grid, DM_BF_THREADS, 0, p->stream>>>(                                   \
        p->btrec, p->bvrec, pt, p->n_faces, p->gd, p->ix_begin, p->ix_end, rps, tau_b_eff, n_tab, p->kappa, p->band_z, p->part)
#define DM_LAUNCH_BF(MODE, SEG)                                                                                          \
    do {                                                                                                                 \
        if (p->band_on) DM_LAUNCH_BF2(MODE, SEG, true); else DM_LAUNCH_BF2(MODE, SEG, false);                            \
    } while (0)
        if (p->mode == DM_SURFACE) {
            if (seg == 8) DM_LAUNCH_BF(1, 8); else if (seg == 16) DM_LAUNCH_BF(1, 16); else DM_LAUNCH_BF(1, 32);
        } else {
            if (seg == 8) DM_LAUNCH_BF(0, 8); else if (seg == 16) DM_LAUNCH_BF(0, 16); else DM_LAUNCH_BF(0, 32);
        }
#undef DM_LAUNCH_BF2
#undef DM_LAUNCH_BF
    } else {
        if ((rc = run_geometry(p, vertices_dev))) return rc;
        dm_k_backward_robust<<<grid, 128, 0, p->stream>>>(p->rec, p->n_faces, p->gd, p->mode, p->ix_begin, p->ix_end, rps,
                                                          (const float2*)G_dev, p->part);
    }
    rc = check_launch(p);
    if (rc) return rc;
    stage_end(p, 0);
    const double *area_total = nullptr, *sdot = nullptr;
    if (p->normalise) {
        // eq. 13's second term needs |Lambda| and sum_k Re(conj(G) F): the caller's spectrum u = F/|Lambda| of these vertices
        // (then the dot product is taken with u), or one raw forward of these vertices
        const long long nk = (long long)n_k_of(p);
        if (!p->dot_part && cudaMalloc(&p->dot_part, (DM_DOT_BLOCKS + 1) * sizeof(double)) != cudaSuccess) return DM_ERR_ALLOC;
        const float2* Fdot = F_reuse;
        if (!Fdot) {
            if (!p->spec3 && cudaMalloc(&p->spec3, (size_t)nk * sizeof(float2)) != cudaSuccess) return DM_ERR_ALLOC;
            p->F_valid = false;
            if ((rc = run_forward_raw(p, vertices_dev, (float*)p->spec3))) return rc;
            Fdot = p->spec3;
        }
        dm_k_dot_partial<<<DM_DOT_BLOCKS, 256, 0, p->stream>>>((const float2*)G_dev, Fdot, nk, p->dot_part);
        if ((rc = check_launch(p))) return rc;
        dm_k_dot_final<<<1, DM_DOT_BLOCKS, 0, p->stream>>>(p->dot_part, p->dot_part + DM_DOT_BLOCKS);
        if ((rc = check_launch(p))) return rc;
        area_total = p->dc_total;
        sdot = p->dot_part + DM_DOT_BLOCKS;
    }
    stage_begin(p, 3);
    int n_split_left = n_split;
    if (n_split > 4) {   // many splits (small meshes): sum them with 13x the threads first
        dm_k_sum_splits<<<dim3((p->n_faces + 127) / 128, DM_BWD_NSUM), 128, 0, p->stream>>>(p->part, p->n_faces, n_split);
        if ((rc = check_launch(p))) return rc;
        n_split_left = 1;
    }
    dm_k_corner_grads<<<(p->n_faces + 127) / 128, 128, 0, p->stream>>>(vertices_dev, p->faces, p->n_faces, p->mode,
                                                                       n_split_left, p->part, (const float2*)G_dev,
                                                                       p->ix_begin == 0 ? 1 : 0, area_total, sdot, F_reuse != nullptr ? 1 : 0, p->gd.face_w,
                                                                       p->corner);
    rc = check_launch(p);
    if (rc) return rc;
    dm_k_vertex_gather<<<(p->n_vertices + 127) / 128, 128, 0, p->stream>>>(p->csr_off, p->csr_corner, p->n_vertices,
                                                                           p->corner, dv_dev);
    rc = check_launch(p);
    stage_end(p, 3);
    return rc;
}

int run_spectrum_to_image(dm_plan* p, const float* F_dev, const DmPsfDev& psf, float* image_dev)
{
    const size_t nk = n_k_of(p);
    stage_begin(p, 1);
    dm_k_psf_multiply<<<(unsigned)((nk + 255) / 256), 256, 0, p->stream>>>((const float2*)F_dev, p->gd, psf, p->spec);
    int rc = check_launch(p);
    stage_end(p, 1);
    if (rc) return rc;
    stage_begin(p, 2);
    if (cufftExecC2C(p->fft_xy, (cufftComplex*)p->spec, (cufftComplex*)p->spec, CUFFT_INVERSE) != CUFFT_SUCCESS)
        return DM_ERR_CUFFT;
    dm_k_drop_selfconj_imag<<<(p->gd.nx * p->gd.ny + 255) / 256, 256, 0, p->stream>>>(p->spec, p->gd);
    rc = check_launch(p);
    if (rc) return rc;
    if (cufftExecC2R(p->fft_z, (cufftComplex*)p->spec, image_dev) != CUFFT_SUCCESS) return DM_ERR_CUFFT;
    stage_end(p, 2);
    return DM_OK;
}

int run_image_to_cotangent(dm_plan* p, const float* dimage_dev, const DmPsfDev& psf, float* G_dev)
{
    const size_t nk = n_k_of(p);
    stage_begin(p, 2);
    if (cufftExecR2C(p->fft_r2c, (cufftReal*)dimage_dev, (cufftComplex*)p->spec) != CUFFT_SUCCESS) return DM_ERR_CUFFT;
    stage_end(p, 2);
    stage_begin(p, 1);
    dm_k_psf_adjoint<<<(unsigned)((nk + 255) / 256), 256, 0, p->stream>>>(p->spec, p->gd, psf, (float2*)G_dev);
    int rc = check_launch(p);
    stage_end(p, 1);
    return rc;
}

}  // namespace

extern "C" {

int dm_version(void) { return DM_VERSION; }

const char* dm_error_string(int code)
{
    const int i = -code;
    return (i >= 0 && i <= 7) ? kErr[i] : "unknown error";
}

int dm_plan_create(dm_plan** out, const dm_grid* grid, int mode, int32_t n_vertices, int32_t n_faces,
                   const int32_t* faces_dev, void* cuda_stream)
{
    if (!out) return DM_ERR_INVALID_ARG;
    *out = nullptr;
    if (!grid || !faces_dev || n_vertices <= 0 || n_faces <= 0 || (mode != DM_VOLUME && mode != DM_SURFACE))
        return DM_ERR_INVALID_ARG;
    for (int d = 0; d < 3; ++d)
        if (grid->n[d] <= 0 || grid->n[d] > 4096 || !(grid->spacing[d] > 0.f) || !std::isfinite(grid->spacing[d]) ||
            !std::isfinite(grid->origin[d]))
            return DM_ERR_INVALID_ARG;
    if (grid->n[2] % 2 != 0) return DM_ERR_INVALID_ARG;
    if ((long long)n_faces * 3 > 0x7fffffffLL) return DM_ERR_INVALID_ARG;

    dm_plan* p = new (std::nothrow) dm_plan();
    if (!p) return DM_ERR_ALLOC;
    p->grid = *grid;
    p->mode = mode;
    p->n_vertices = n_vertices;
    p->n_faces = n_faces;
    p->stream = (cudaStream_t)cuda_stream;
    p->gd.nx = grid->n[0];
    p->gd.ny = grid->n[1];
    p->gd.nz = grid->n[2];
    p->gd.nzh = grid->n[2] / 2 + 1;
    for (int d = 0; d < 3; ++d) {
        const double L = (double)grid->n[d] * (double)grid->spacing[d];
        p->gd.kstep[d] = (float)(2.0 * M_PI / L);
        p->gd.inv_len[d] = 1.0 / L;
    }
    for (int i = 0; i < 6; ++i) p->gd.band_cov[i] = 0.f;
    p->gd.band_lim = INFINITY;
    p->gd.nzb = p->gd.nzh;
    p->gd.band_slots = nullptr;
    p->gd.n_band_slots = 0;
    p->gd.face_w = nullptr;
    {
        double lmax = 0.0;
        for (int dd = 0; dd < 3; ++dd) lmax = std::max(lmax, (double)grid->n[dd] * (double)grid->spacing[dd]);
        p->gd.edge_fix = (float)(1073741824.0 / (lmax * lmax));   // squared edges in units of 2^-30 L_max^2
        p->gd.inv_edge_norm = (float)(1.0 / (3.0 * (double)n_faces * (double)p->gd.edge_fix));
    }
    p->ix_begin = 0;
    p->ix_end = p->gd.nx;
    // gap-product threshold of the forward fast path: one excluded-or-not pair may cost ~1e-6 (sum|d|)/tau of ONE
    // triangle's weight, i.e. ~1e-5/(n_T tau) of |F(0)|; tau n_T = 0.5 keeps the measured maximum over the grid near
    // 2e-5 |F(0)|, a fifth of the tolerance
    p->tau = (float)std::min(1e-2, std::max(5e-6, 0.5 / (double)n_faces));

    int rc = DM_OK;
    int dev = 0;
    std::vector<int32_t> faces_h, off, cor, fill;
    do {
        if (cudaGetDevice(&dev) != cudaSuccess ||
            cudaDeviceGetAttribute(&p->n_sm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) { rc = DM_ERR_CUDA; break; }
        try {
            faces_h.resize((size_t)n_faces * 3);
            off.assign((size_t)n_vertices + 1, 0);
            cor.resize((size_t)n_faces * 3);
        } catch (...) { rc = DM_ERR_ALLOC; break; }
        if (cudaMemcpyAsync(faces_h.data(), faces_dev, faces_h.size() * sizeof(int32_t), cudaMemcpyDeviceToHost,
                            p->stream) != cudaSuccess || cudaStreamSynchronize(p->stream) != cudaSuccess) { rc = DM_ERR_CUDA; break; }
        bool bad = false;
        for (size_t i = 0; i < faces_h.size(); ++i) {
            const int32_t v = faces_h[i];
            if (v < 0 || v >= n_vertices) { bad = true; break; }
            off[(size_t)v + 1]++;
        }
        if (bad) { rc = DM_ERR_BAD_MESH; break; }
        // CSR vertex -> corner (3*face+corner), ascending corner id per vertex: the vertex star v* of eq. 13
        for (int32_t v = 0; v < n_vertices; ++v) off[(size_t)v + 1] += off[v];
        try { fill.assign(off.begin(), off.end() - 1); } catch (...) { rc = DM_ERR_ALLOC; break; }
        for (size_t i = 0; i < faces_h.size(); ++i) cor[(size_t)fill[faces_h[i]]++] = (int32_t)i;

        // connected components of the faces (shared vertices; union-find), used to classify per-face weights
        try {
            std::vector<int32_t> parent((size_t)n_vertices);
            for (int32_t v = 0; v < n_vertices; ++v) parent[v] = v;
            auto find = [&](int32_t a) {
                while (parent[a] != a) {
                    parent[a] = parent[parent[a]];
                    a = parent[a];
                }
                return a;
            };
            for (int32_t t = 0; t < n_faces; ++t) {
                const int32_t a = find(faces_h[3 * (size_t)t]);
                for (int j = 1; j < 3; ++j) {
                    const int32_t b = find(faces_h[3 * (size_t)t + j]);
                    if (b != a) parent[b] = a;
                }
            }
            p->face_comp.resize((size_t)n_faces);
            for (int32_t t = 0; t < n_faces; ++t) p->face_comp[t] = find(faces_h[3 * (size_t)t]);
        } catch (...) { rc = DM_ERR_ALLOC; break; }

        try { p->faces_host = faces_h; } catch (...) { rc = DM_ERR_ALLOC; break; }
        const size_t nk = n_k_of(p);
        // k-splits of the backward: a small mesh has few triangle blocks, so it needs many splits to fill the machine
        // (up to 48 CTAs per SM slot), within 64 M floats of partial sums
        p->n_split_max = dm_backward_split_max(p->n_sm, DM_BWD_SPLIT_TARGET, DM_BWD_NSUM, n_faces, (long long)p->gd.nx * p->gd.ny);
        if (cudaMalloc(&p->faces, faces_h.size() * sizeof(int32_t)) != cudaSuccess ||
            cudaMalloc(&p->csr_off, off.size() * sizeof(int32_t)) != cudaSuccess ||
            cudaMalloc(&p->csr_corner, cor.size() * sizeof(int32_t)) != cudaSuccess ||
            cudaMalloc(&p->rec, (size_t)n_faces * 4 * sizeof(float4)) != cudaSuccess ||
            cudaMalloc(&p->part, (size_t)p->n_split_max * DM_BWD_NSUM * n_faces * sizeof(float)) != cudaSuccess ||
            cudaMalloc(&p->corner, (size_t)n_faces * 9 * sizeof(float)) != cudaSuccess ||
            cudaMalloc(&p->spec, nk * sizeof(float2)) != cudaSuccess) { rc = DM_ERR_ALLOC; break; }
        if (cudaMemcpyAsync(p->faces, faces_h.data(), faces_h.size() * sizeof(int32_t), cudaMemcpyHostToDevice, p->stream) != cudaSuccess ||
            cudaMemcpyAsync(p->csr_off, off.data(), off.size() * sizeof(int32_t), cudaMemcpyHostToDevice, p->stream) != cudaSuccess ||
            cudaMemcpyAsync(p->csr_corner, cor.data(), cor.size() * sizeof(int32_t), cudaMemcpyHostToDevice, p->stream) != cudaSuccess ||
            cudaStreamSynchronize(p->stream) != cudaSuccess) { rc = DM_ERR_CUDA; break; }
        // strip walk for the fast forward kernel; chunks so that (k-blocks x chunks) fills the machine several times
        {
            const int n_yruns = (p->gd.ny + DM_K - 1) / DM_K;
            const long long kblocks = ((long long)p->gd.nx * n_yruns * p->gd.nzh + DM_FAST_THREADS - 1) / DM_FAST_THREADS;
            const long long slots = (long long)p->n_sm * 4;
            long long want = (6 * slots + kblocks - 1) / kblocks;
            // a chunk costs two flush records and one row of partial spectra: at least DM_FAST_MIN_CHUNK faces each.  Large
            // meshes fill the machine with few chunks of whole tiles; a small mesh on a small grid (an
            // 80-triangle sphere; :261: 10 000 such steps) needs the short chunks to reach every SM
            want = std::min<long long>(want, std::max<long long>(1, n_faces / DM_FAST_MIN_CHUNK));
            want = std::max<long long>(1, std::min<long long>(want, 64));
            DmStripRecords sr;
            try { sr = dm_build_strips(faces_h.data(), n_faces, n_vertices, (int)want); } catch (...) { rc = DM_ERR_ALLOC; break; }
            p->st_n_rec = (int)sr.fid.size();
            p->st_n_chunks = (int)sr.chunk_off.size() - 1;
            const size_t nb = (size_t)p->st_n_rec * sizeof(int32_t);
            if (cudaMalloc(&p->st_new, nb) != cudaSuccess || cudaMalloc(&p->st_prev, nb) != cudaSuccess ||
                cudaMalloc(&p->st_ret, nb) != cudaSuccess || cudaMalloc(&p->st_fid, nb) != cudaSuccess ||
                cudaMalloc(&p->st_chunk_off, sr.chunk_off.size() * sizeof(int32_t)) != cudaSuccess ||
                cudaMalloc(&p->st_rec, (size_t)p->st_n_rec * 3 * sizeof(float4)) != cudaSuccess ||
                cudaMalloc(&p->fwd_part, (size_t)p->st_n_chunks * nk * sizeof(float2)) != cudaSuccess ||
                cudaMalloc(&p->hmax2, 16) != cudaSuccess ||
                cudaMalloc(&p->dc_part, DM_DC_BLOCKS * sizeof(double)) != cudaSuccess ||
                cudaMalloc(&p->dc_total, sizeof(double)) != cudaSuccess) { rc = DM_ERR_ALLOC; break; }
            if (cudaMemcpyAsync(p->st_new, sr.vid_new.data(), nb, cudaMemcpyHostToDevice, p->stream) != cudaSuccess ||
                cudaMemcpyAsync(p->st_prev, sr.vid_prev.data(), nb, cudaMemcpyHostToDevice, p->stream) != cudaSuccess ||
                cudaMemcpyAsync(p->st_ret, sr.vid_ret.data(), nb, cudaMemcpyHostToDevice, p->stream) != cudaSuccess ||
                cudaMemcpyAsync(p->st_fid, sr.fid.data(), nb, cudaMemcpyHostToDevice, p->stream) != cudaSuccess ||
                cudaMemcpyAsync(p->st_chunk_off, sr.chunk_off.data(), sr.chunk_off.size() * sizeof(int32_t),
                                cudaMemcpyHostToDevice, p->stream) != cudaSuccess ||
                cudaStreamSynchronize(p->stream) != cudaSuccess) { rc = DM_ERR_CUDA; break; }
        }
        // patches of 32 triangles for the fast backward kernel (shared vertex phases), padded to whole CTAs
        {
            DmPatches pp;
            try {
                pp = dm_build_patches(faces_h.data(), n_faces, n_vertices);
                while ((pp.face.size() % DM_BF_THREADS) != 0) {   // padding patch: idle lanes, no vertices
                    pp.face.insert(pp.face.end(), DM_PATCH_FACES, -1);
                    pp.loc.insert(pp.loc.end(), DM_PATCH_FACES, 0u);
                    pp.vid.insert(pp.vid.end(), DM_PATCH_MAXV, -1);
                }
            } catch (...) { rc = DM_ERR_ALLOC; break; }
            p->pt_lanes = (int)pp.face.size();
            const size_t nl = pp.face.size();
            if (cudaMalloc(&p->pt_face, nl * sizeof(int32_t)) != cudaSuccess ||
                cudaMalloc(&p->pt_loc, nl * sizeof(uint32_t)) != cudaSuccess ||
                cudaMalloc(&p->pt_vid, pp.vid.size() * sizeof(int32_t)) != cudaSuccess ||
                cudaMalloc(&p->btrec, nl * DM_BF_TREC * sizeof(float4)) != cudaSuccess ||
                cudaMalloc(&p->bvrec, nl * DM_BF_VREC * sizeof(float4)) != cudaSuccess) { rc = DM_ERR_ALLOC; break; }
            if (cudaMemcpyAsync(p->pt_face, pp.face.data(), nl * sizeof(int32_t), cudaMemcpyHostToDevice, p->stream) != cudaSuccess ||
                cudaMemcpyAsync(p->pt_loc, pp.loc.data(), nl * sizeof(uint32_t), cudaMemcpyHostToDevice, p->stream) != cudaSuccess ||
                cudaMemcpyAsync(p->pt_vid, pp.vid.data(), pp.vid.size() * sizeof(int32_t), cudaMemcpyHostToDevice, p->stream) != cudaSuccess ||
                cudaStreamSynchronize(p->stream) != cudaSuccess) { rc = DM_ERR_CUDA; break; }
        }
        bool ok = true;
        for (int i = 0; i < 8; ++i) ok = ok && (cudaEventCreate(&p->ev[i]) == cudaSuccess);
        if (!ok) { rc = DM_ERR_CUDA; break; }
        p->ev_ok = true;
    } while (0);
    if (rc != DM_OK) {
        dm_plan_destroy(p);
        cudaGetLastError();
        return rc;
    }
    *out = p;
    return DM_OK;
}

int dm_plan_set_stream(dm_plan* p, void* cuda_stream)
{
    if (!p) return DM_ERR_INVALID_ARG;
    p->stream = (cudaStream_t)cuda_stream;
    if (p->have_fft && (cufftSetStream(p->fft_xy, p->stream) != CUFFT_SUCCESS || cufftSetStream(p->fft_z, p->stream) != CUFFT_SUCCESS ||
                        cufftSetStream(p->fft_r2c, p->stream) != CUFFT_SUCCESS))
        return DM_ERR_CUFFT;
    return DM_OK;
}

int dm_plan_set_slab(dm_plan* p, int32_t ix_begin, int32_t ix_end)
{
    if (!p || ix_begin < 0 || ix_end > p->gd.nx || ix_begin >= ix_end) return DM_ERR_INVALID_ARG;
    p->ix_begin = ix_begin;
    p->ix_end = ix_end;
    p->F_valid = false;
    return DM_OK;
}

int dm_plan_set_face_weights(dm_plan* p, const float* weights_dev)
{
    if (!p) return DM_ERR_INVALID_ARG;
    p->F_valid = false;
    if (!weights_dev) {
        p->gd.face_w = nullptr;
        p->weights_robust = false;
        return DM_OK;
    }
    // classify on the host (this call synchronises the stream): the fast kernels' flag thresholds are validated, against
    // the tolerance 1e-4 |F(0)|, for weights of one sign that -- in volume mode -- are constant on every connected
    // component (regions of different density); anything else (mixed signs: F(0) cancels and stops being the scale of the
    // spectrum; weights varying inside a component in volume mode: the rounding errors of a shared edge no longer cancel
    // between its two faces) is evaluated pair by pair through the robust branches
    std::vector<float> wh;
    try { wh.resize((size_t)p->n_faces); } catch (...) { return DM_ERR_ALLOC; }
    if (cudaMemcpyAsync(wh.data(), weights_dev, wh.size() * sizeof(float), cudaMemcpyDeviceToHost, p->stream) != cudaSuccess ||
        cudaStreamSynchronize(p->stream) != cudaSuccess)
        return DM_ERR_CUDA;
    bool pos = false, neg = false, split = false;
    std::vector<float> comp_w;
    std::vector<char> comp_seen;
    try {
        if (p->mode == DM_VOLUME) {
            comp_w.assign((size_t)p->n_vertices, 0.f);
            comp_seen.assign((size_t)p->n_vertices, 0);
        }
    } catch (...) { return DM_ERR_ALLOC; }
    for (int32_t t = 0; t < p->n_faces; ++t) {
        const float w = wh[t];
        if (!std::isfinite(w)) return DM_ERR_INVALID_ARG;
        pos = pos || w > 0.f;
        neg = neg || w < 0.f;
        if (p->mode == DM_VOLUME) {
            const int32_t c = p->face_comp[t];
            if (!comp_seen[c]) {
                comp_seen[c] = 1;
                comp_w[c] = w;
            } else if (comp_w[c] != w) {
                split = true;
            }
        }
    }
    if (!p->face_w && cudaMalloc(&p->face_w, (size_t)p->n_faces * sizeof(float)) != cudaSuccess) return DM_ERR_ALLOC;
    if (cudaMemcpyAsync(p->face_w, weights_dev, (size_t)p->n_faces * sizeof(float), cudaMemcpyDeviceToDevice, p->stream) !=
        cudaSuccess)
        return DM_ERR_CUDA;
    p->gd.face_w = p->face_w;
    p->weights_robust = (pos && neg) || split;
    return DM_OK;
}

int dm_plan_update_face_weights(dm_plan* p, const float* weights_dev, int32_t robust)
{
    if (!p || !weights_dev || (robust != 0 && robust != 1)) return DM_ERR_INVALID_ARG;
    p->F_valid = false;
    if (!p->face_w && cudaMalloc(&p->face_w, (size_t)p->n_faces * sizeof(float)) != cudaSuccess) return DM_ERR_ALLOC;
    if (cudaMemcpyAsync(p->face_w, weights_dev, (size_t)p->n_faces * sizeof(float), cudaMemcpyDeviceToDevice, p->stream) !=
        cudaSuccess)
        return DM_ERR_CUDA;
    p->gd.face_w = p->face_w;
    p->weights_robust = robust != 0;   // the caller's word: nothing is read back
    return DM_OK;
}

int dm_plan_set_narrow_band(dm_plan* p, const float* psf_cov_host, float cutoff)
{
    if (!p) return DM_ERR_INVALID_ARG;
    p->F_valid = false;
    if (!psf_cov_host) {
        p->band_on = false;
        p->gd.band_lim = INFINITY;
        p->gd.nzb = p->gd.nzh;
        p->gd.band_slots = nullptr;
        p->gd.n_band_slots = 0;
        return DM_OK;
    }
    if (!(cutoff > 0.f) || !(cutoff < 1.f)) return DM_ERR_INVALID_ARG;
    for (int i = 0; i < 6; ++i)
        if (!std::isfinite(psf_cov_host[i])) return DM_ERR_INVALID_ARG;
    // Everything is built beside the plan's current band and committed at the end: a failed call leaves the plan as it was.
    DmGridDev g = p->gd;
    for (int i = 0; i < 6; ++i) g.band_cov[i] = psf_cov_host[i];
    g.band_lim = std::log(1.0f / cutoff);
    // extent of the band ellipsoid along z: k_z^2 <= 2 L (B^-1)_zz; two frequencies of margin, the whole axis when B is
    // not positive definite
    {
        const double xx = psf_cov_host[0], yy = psf_cov_host[1], zz = psf_cov_host[2], xy = psf_cov_host[3],
                     xz = psf_cov_host[4], yz = psf_cov_host[5];
        const double det = xx * (yy * zz - yz * yz) - xy * (xy * zz - yz * xz) + xz * (xy * yz - yy * xz);
        const double cof = xx * yy - xy * xy;
        g.nzb = g.nzh;
        if (det > 0.0 && cof > 0.0 && xx > 0.0) {
            const double kz_max = std::sqrt(2.0 * (double)g.band_lim * cof / det);
            const double nz_max = kz_max / (double)g.kstep[2];
            if (nz_max + 3.0 < (double)g.nzh) g.nzb = (int)nz_max + 3;
        }
    }
    const int n_rows = g.nx * g.ny;
    g.band_slots = nullptr;   // the row intervals are computed with the band test alone
    g.n_band_slots = 0;
    int2* band_z_new = nullptr;
    uint32_t* slots_new = nullptr;
    int rc = DM_OK;
    long long count = 0;
    std::vector<int2> bz;
    std::vector<uint32_t> slots;
    do {
        if (cudaMalloc(&band_z_new, (size_t)n_rows * sizeof(int2)) != cudaSuccess) { rc = DM_ERR_ALLOC; break; }
        dm_k_band_rows<<<(n_rows + 127) / 128, 128, 0, p->stream>>>(g, band_z_new);
        if ((rc = check_launch(p))) break;
        // the forward kernel's thread list: every (i_x, run of DM_K signed y-frequencies, i_z) with a frequency in the band
        try { bz.resize((size_t)n_rows); } catch (...) { rc = DM_ERR_ALLOC; break; }
        if (cudaMemcpyAsync(bz.data(), band_z_new, (size_t)n_rows * sizeof(int2), cudaMemcpyDeviceToHost, p->stream) != cudaSuccess ||
            cudaStreamSynchronize(p->stream) != cudaSuccess) { rc = DM_ERR_CUDA; break; }
        for (const int2& b : bz) count += std::max(0, b.y - b.x);
        const int ny = g.ny, n_yruns = (ny + DM_K - 1) / DM_K;
        if (g.nx <= 4096 && n_yruns <= 2048 && g.nzh <= 512) {
            try {
                for (int ix = 0; ix < g.nx; ++ix)
                    for (int yrun = 0; yrun < n_yruns; ++yrun) {
                        int lo = g.nzh, hi = 0;
                        for (int j = 0; j < DM_K; ++j) {
                            const int nys = -(ny / 2) + yrun * DM_K + j;
                            if (nys > (ny - 1) / 2) break;
                            const int2 b = bz[(size_t)ix * ny + (nys < 0 ? nys + ny : nys)];
                            if (b.y > b.x) {
                                lo = std::min(lo, b.x);
                                hi = std::max(hi, b.y);
                            }
                        }
                        for (int iz = lo; iz < hi; ++iz) slots.push_back(((uint32_t)ix << 20) | ((uint32_t)yrun << 9) | (uint32_t)iz);
                    }
            } catch (...) { rc = DM_ERR_ALLOC; break; }
            if (!slots.empty()) {
                if (cudaMalloc(&slots_new, slots.size() * sizeof(uint32_t)) != cudaSuccess) { rc = DM_ERR_ALLOC; break; }
                if (cudaMemcpyAsync(slots_new, slots.data(), slots.size() * sizeof(uint32_t), cudaMemcpyHostToDevice, p->stream) !=
                        cudaSuccess ||
                    cudaStreamSynchronize(p->stream) != cudaSuccess) { rc = DM_ERR_CUDA; break; }
                g.band_slots = slots_new;
                g.n_band_slots = (int)slots.size();
            }
        }
    } while (0);
    if (rc != DM_OK) {
        cudaFree(band_z_new);
        cudaFree(slots_new);
        cudaGetLastError();
        return rc;
    }
    // commit (the stream is idle: the copies above were synchronised)
    cudaFree(p->band_z);
    cudaFree(p->band_slots);
    p->band_z = band_z_new;
    p->band_slots = slots_new;
    p->gd = g;
    p->band_count = count;
    p->band_on = true;
    return DM_OK;
}

int dm_plan_set_option(dm_plan* p, int option, double value)
{
    if (!p) return DM_ERR_INVALID_ARG;
    if (option != DM_OPT_REUSE_SPECTRUM) p->F_valid = false;
    switch (option) {
        case DM_OPT_REUSE_SPECTRUM:
            if (value != 0.0 && value != 1.0) return DM_ERR_INVALID_ARG;
            p->reuse_F = value == 1.0;
            return DM_OK;
        case DM_OPT_FORWARD_PATH:
            if (value != 0.0 && value != 1.0) return DM_ERR_INVALID_ARG;
            p->fwd_path = (int)value;
            return DM_OK;
        case DM_OPT_BACKWARD_PATH:
            if (value != 0.0 && value != 1.0) return DM_ERR_INVALID_ARG;
            p->bwd_path = (int)value;
            return DM_OK;
        case DM_OPT_TAU:      // 0 is allowed: only exactly vanishing gap products then leave the fast path
            if (!(value >= 0.0) || !std::isfinite(value)) return DM_ERR_INVALID_ARG;
            p->tau = (float)value;
            return DM_OK;
        case DM_OPT_AREA_NORMALISED:
            if ((value != 0.0 && value != 1.0) || (value == 1.0 && p->mode != DM_SURFACE)) return DM_ERR_INVALID_ARG;
            p->normalise = value == 1.0;
            return DM_OK;
        case DM_OPT_TAU_BWD:
            if (!(value >= 0.0) || !std::isfinite(value)) return DM_ERR_INVALID_ARG;
            p->tau_b = (float)value;
            return DM_OK;
        default:
            return DM_ERR_INVALID_ARG;
    }
}

int dm_mesh_ft_forward(dm_plan* p, const float* vertices_dev, float* F_dev)
{
    if (!p || !vertices_dev || !F_dev) return DM_ERR_INVALID_ARG;
    p->F_valid = false;   // the plan's total area / volume now belongs to these vertices
    stage_reset(p);
    stage_begin(p, 0);
    const int rc = run_forward(p, vertices_dev, F_dev);
    stage_end(p, 0);
    return rc;
}

int dm_mesh_ft_backward(dm_plan* p, const float* vertices_dev, const float* dL_dF_dev, float* dL_dvertices_dev)
{
    if (!p || !vertices_dev || !dL_dF_dev || !dL_dvertices_dev) return DM_ERR_INVALID_ARG;
    stage_reset(p);
    stage_begin(p, 0);
    return run_backward(p, vertices_dev, dL_dF_dev, dL_dvertices_dev);
}

int dm_mesh_ft_backward_with_spectrum(dm_plan* p, const float* vertices_dev, const float* dL_dF_dev, const float* F_dev,
                                      float* dL_dvertices_dev)
{
    if (!p || !vertices_dev || !dL_dF_dev || !F_dev || !dL_dvertices_dev) return DM_ERR_INVALID_ARG;
    stage_reset(p);
    stage_begin(p, 0);
    return run_backward(p, vertices_dev, dL_dF_dev, dL_dvertices_dev, p->normalise ? (const float2*)F_dev : nullptr);
}

int dm_spectrum_to_image(dm_plan* p, const float* F_dev, const float* psf_cov_host, float* image_dev)
{
    if (!p || !F_dev || !image_dev) return DM_ERR_INVALID_ARG;
    DmPsfDev psf;
    int rc = make_psf(p, psf_cov_host, &psf);
    if (rc) return rc;
    if ((rc = ensure_fft(p))) return rc;
    stage_reset(p);
    return run_spectrum_to_image(p, F_dev, psf, image_dev);
}

int dm_image_to_spectrum_cotangent(dm_plan* p, const float* dL_dimage_dev, const float* psf_cov_host, float* G_dev)
{
    if (!p || !dL_dimage_dev || !G_dev) return DM_ERR_INVALID_ARG;
    DmPsfDev psf;
    int rc = make_psf(p, psf_cov_host, &psf);
    if (rc) return rc;
    if ((rc = ensure_fft(p))) return rc;
    stage_reset(p);
    return run_image_to_cotangent(p, dL_dimage_dev, psf, G_dev);
}

int dm_render(dm_plan* p, const float* vertices_dev, const float* psf_cov_host, float* image_dev)
{
    if (!p || !vertices_dev || !image_dev) return DM_ERR_INVALID_ARG;
    if (p->ix_begin != 0 || p->ix_end != p->gd.nx) return DM_ERR_INVALID_ARG;
    DmPsfDev psf;
    int rc = make_psf(p, psf_cov_host, &psf);
    if (rc) return rc;
    if ((rc = ensure_fft(p))) return rc;
    stage_reset(p);
    if (!p->spec3 && cudaMalloc(&p->spec3, n_k_of(p) * sizeof(float2)) != cudaSuccess) return DM_ERR_ALLOC;
    p->F_valid = false;
    stage_begin(p, 0);
    rc = run_forward(p, vertices_dev, (float*)p->spec3);   // F stays in the plan for dm_render_backward (DM_OPT_REUSE_SPECTRUM)
    stage_end(p, 0);
    if (rc) return rc;
    rc = run_spectrum_to_image(p, (const float*)p->spec3, psf, image_dev);
    p->F_valid = rc == DM_OK;
    return rc;
}

int dm_render_backward(dm_plan* p, const float* vertices_dev, const float* psf_cov_host, const float* dL_dimage_dev,
                       float* dL_dvertices_dev, float* dL_dpsf_cov_host)
{
    if (!p || !vertices_dev || !dL_dimage_dev || !dL_dvertices_dev) return DM_ERR_INVALID_ARG;
    if (p->ix_begin != 0 || p->ix_end != p->gd.nx) return DM_ERR_INVALID_ARG;
    DmPsfDev psf;
    int rc = make_psf(p, psf_cov_host, &psf);
    if (rc) return rc;
    if ((rc = ensure_fft(p))) return rc;
    const bool reuse = p->reuse_F && (dL_dpsf_cov_host || p->normalise);
    if (reuse && !p->F_valid) return DM_ERR_INVALID_ARG;   // no dm_render spectrum to reuse (or something changed since)
    if (dL_dpsf_cov_host) {
        const size_t nk = n_k_of(p);
        if (!p->spec3 && cudaMalloc(&p->spec3, nk * sizeof(float2)) != cudaSuccess) return DM_ERR_ALLOC;
        if (!p->psfg_part && cudaMalloc(&p->psfg_part, DM_PSFG_BLOCKS * 6 * sizeof(double)) != cudaSuccess) return DM_ERR_ALLOC;
        if (!p->psfg_out && cudaMalloc(&p->psfg_out, 6 * sizeof(float)) != cudaSuccess) return DM_ERR_ALLOC;
    }
    stage_reset(p);
    rc = run_image_to_cotangent(p, dL_dimage_dev, psf, (float*)p->spec2);   // leaves R = rfft3(dL/dimage) in p->spec
    if (rc) return rc;
    stage_begin(p, 0);
    rc = run_backward(p, vertices_dev, (const float*)p->spec2, dL_dvertices_dev, reuse ? p->spec3 : nullptr);
    if (rc || !dL_dpsf_cov_host) return rc;
    // PSF-parameter gradient: needs the forward spectrum F of these vertices -- the one dm_render left in the plan
    // (DM_OPT_REUSE_SPECTRUM), else recomputed (one forward mesh FT)
    if (!reuse) {
        p->F_valid = false;
        if ((rc = run_forward(p, vertices_dev, (float*)p->spec3))) return rc;
    }
    dm_k_psf_grad_partial<<<DM_PSFG_BLOCKS, 256, 0, p->stream>>>(p->spec, p->spec3, p->gd, psf, p->psfg_part);
    if ((rc = check_launch(p))) return rc;
    dm_k_psf_grad_final<<<1, DM_PSFG_BLOCKS, 0, p->stream>>>(p->psfg_part, p->psfg_out);
    if ((rc = check_launch(p))) return rc;
    if (cudaMemcpyAsync(dL_dpsf_cov_host, p->psfg_out, 6 * sizeof(float), cudaMemcpyDeviceToHost, p->stream) != cudaSuccess ||
        cudaStreamSynchronize(p->stream) != cudaSuccess)
        return DM_ERR_CUDA;
    return DM_OK;
}

int dm_plan_stage_ms(dm_plan* p, float ms[4])
{
    if (!p || !ms) return DM_ERR_INVALID_ARG;
    if (cudaStreamSynchronize(p->stream) != cudaSuccess) return DM_ERR_CUDA;
    for (int s = 0; s < 4; ++s) {
        ms[s] = 0.f;
        if (p->stage_ran[s] && cudaEventElapsedTime(&ms[s], p->ev[2 * s], p->ev[2 * s + 1]) != cudaSuccess) return DM_ERR_CUDA;
    }
    return DM_OK;
}

int64_t dm_plan_launch_count(const dm_plan* p) { return p ? p->launches : 0; }

int dm_plan_paths_used(const dm_plan* p, int32_t paths[2])
{
    if (!p || !paths) return DM_ERR_INVALID_ARG;
    paths[0] = p->last_fwd_path;
    paths[1] = p->last_bwd_path;
    return DM_OK;
}

void dm_plan_destroy(dm_plan* p)
{
    if (!p) return;
    if (p->have_xy) cufftDestroy(p->fft_xy);
    if (p->have_z) cufftDestroy(p->fft_z);
    if (p->have_r2c) cufftDestroy(p->fft_r2c);
    cudaFree(p->faces);
    cudaFree(p->csr_off);
    cudaFree(p->csr_corner);
    cudaFree(p->rec);
    cudaFree(p->pt_face);
    cudaFree(p->pt_vid);
    cudaFree(p->pt_loc);
    cudaFree(p->btrec);
    cudaFree(p->bvrec);
    cudaFree(p->part);
    cudaFree(p->corner);
    cudaFree(p->spec);
    cudaFree(p->spec2);
    cudaFree(p->st_new);
    cudaFree(p->st_prev);
    cudaFree(p->st_ret);
    cudaFree(p->st_fid);
    cudaFree(p->st_chunk_off);
    cudaFree(p->st_rec);
    cudaFree(p->fwd_part);
    cudaFree(p->hmax2);
    cudaFree(p->dc_part);
    cudaFree(p->dc_total);
    cudaFree(p->dot_part);
    cudaFree(p->face_w);
    cudaFree(p->band_slots);
    cudaFree(p->band_z);
    cudaFree(p->spec3);
    cudaFree(p->kappa);
    cudaFree(p->psfg_part);
    cudaFree(p->psfg_out);
    if (p->ev_ok)
        for (int i = 0; i < 8; ++i) cudaEventDestroy(p->ev[i]);
    delete p;
}

}  // extern "C"

// ---- shape-optimisation step (eq. 17) -------------------------------------------------------------------
struct dm_shape_state {
    dm_plan* plan = nullptr;
    dm_shape_params prm;
    int n_blocks = 0;                // ceil(n_vertices / DM_SH_THREADS)
    int32_t *adj_off = nullptr, *adj_idx = nullptr;   // CSR of the distinct neighbours of every vertex (L = D - A)
    double *cg_x = nullptr, *cg_y = nullptr, *cg_r = nullptr, *cg_p = nullptr, *cg_Ap = nullptr;
    double *part_a = nullptr, *part_b = nullptr;
    DmCgScalars* cg_sc = nullptr;    // [2]: the scalars of the current and of the next iteration
    int cg_iter_bound = 0;           // iterations after which CG has converged to cg_tol whatever the right-hand side
    int coop_blocks = 0;             // > 0: blocks of the persistent (cooperative) solve; 0: the multi-launch solve
    int* cg_iters = nullptr;         // [2] device: iterations the two solves of the last preconditioning took (persistent solve)
    double* cg_res = nullptr;        // [2] device: relative residual max_c |r|/|b| the two solves ended with (both solve forms)
    double *mom = nullptr, *amax_part = nullptr, *s_next = nullptr;
    DmAdamScalars* adam = nullptr;
    float *image = nullptr, *cot = nullptr, *grad = nullptr;
    double *loss_part = nullptr, *loss = nullptr;
};

namespace {

// x = M^-1 b, M = I + lambda L, for the three columns of b ([n][3], fp32 or fp64), by conjugate gradients on the device
template <typename TB>
int shape_cg_solve(dm_plan* p, dm_shape_state* st, const TB* b_dev, double* x_dev, int which)
{
    const int n = p->n_vertices, nb = st->n_blocks;
    if (st->coop_blocks > 0) {
        // one persistent kernel: grid barriers instead of launches, stops at convergence
        int n_ = n, max_iter = st->prm.cg_max_iter;
        double lambda = (double)st->prm.lambda, tol2_ = (double)st->prm.cg_tol * (double)st->prm.cg_tol;
        int* iters = st->cg_iters + which;
        double* res = st->cg_res + which;
        void* args[] = {(void*)&st->adj_off, (void*)&st->adj_idx, (void*)&n_, (void*)&lambda, (void*)&b_dev, (void*)&x_dev,
                        (void*)&st->cg_r, (void*)&st->cg_p, (void*)&st->cg_Ap, (void*)&st->part_a, (void*)&st->part_b,
                        (void*)&tol2_, (void*)&max_iter, (void*)&iters, (void*)&res};
        if (cudaLaunchCooperativeKernel((const void*)dm_k_cg_persistent<TB>, dim3((unsigned)st->coop_blocks), dim3(DM_SH_THREADS),
                                        args, 0, p->stream) == cudaSuccess)
            return check_launch(p, 1);
        // the device refused the cooperative launch (e.g. it cannot make the whole grid resident right now): the same solve
        // as separate launches, from now on
        cudaGetLastError();
        st->coop_blocks = 0;
    }
    dm_k_cg_init<TB><<<nb, DM_SH_THREADS, 0, p->stream>>>(b_dev, n, x_dev, st->cg_r, st->cg_p, st->part_a);
    dm_k_cg_init_final<<<1, DM_SH_THREADS, 0, p->stream>>>(st->part_a, nb, st->cg_sc);
    int rc = check_launch(p, 2);
    const double tol2 = (double)st->prm.cg_tol * (double)st->prm.cg_tol;
    const int n_iter = std::min(st->prm.cg_max_iter, st->cg_iter_bound);
    for (int it = 0; it < n_iter && rc == DM_OK; ++it) {
        const DmCgScalars* sc = st->cg_sc + (it & 1);
        DmCgScalars* sc_next = st->cg_sc + ((it + 1) & 1);
        dm_k_cg_spmv<<<nb, DM_SH_THREADS, 0, p->stream>>>(st->adj_off, st->adj_idx, n, (double)st->prm.lambda, st->cg_p, st->cg_Ap,
                                                           st->part_a, sc);
        dm_k_cg_update_x<<<nb, DM_SH_THREADS, 0, p->stream>>>(n, st->cg_p, st->cg_Ap, x_dev, st->cg_r, st->part_a, st->part_b, nb, sc);
        dm_k_cg_update_p<<<nb, DM_SH_THREADS, 0, p->stream>>>(n, st->cg_r, st->cg_p, st->part_b, nb, sc, sc_next, tol2);
        rc = check_launch(p, 3);
    }
    if (rc) return rc;
    dm_k_cg_residual<<<1, 1, 0, p->stream>>>(st->cg_sc + (n_iter & 1), st->cg_res + which);
    return check_launch(p);
}

// out = (I + lambda L)^-2 g: two solves (reading R27); the result stays in st->cg_x (fp64)
int shape_precondition(dm_plan* p, dm_shape_state* st, const float* g_dev)
{
    int rc = shape_cg_solve<float>(p, st, g_dev, st->cg_y, 0);
    if (rc) return rc;
    return shape_cg_solve<double>(p, st, st->cg_y, st->cg_x, 1);
}

}  // namespace

extern "C" {

int dm_shape_params_default(dm_shape_params* out)
{
    if (!out) return DM_ERR_INVALID_ARG;
    out->lr = 1e-3f;
    out->lambda = 50.0f;
    out->beta1 = 0.9f;
    out->beta2 = 0.999f;
    out->eps = 1e-8f;
    out->cg_tol = 1e-7f;
    out->cg_max_iter = 400;
    out->solver = 0;
    return DM_OK;
}

int dm_shape_state_create(dm_plan* p, const dm_shape_params* params, dm_shape_state** out)
{
    if (!out) return DM_ERR_INVALID_ARG;
    *out = nullptr;
    if (!p) return DM_ERR_INVALID_ARG;
    dm_shape_params prm;
    dm_shape_params_default(&prm);
    if (params) prm = *params;
    if (!(prm.lr > 0.f) || !(prm.lambda >= 0.f) || !(prm.beta1 >= 0.f && prm.beta1 < 1.f) || !(prm.beta2 >= 0.f && prm.beta2 < 1.f) ||
        !(prm.eps >= 0.f) || !(prm.cg_tol > 0.f) || prm.cg_max_iter < 1 || (prm.solver != 0 && prm.solver != 1) || !std::isfinite(prm.lr) || !std::isfinite(prm.lambda))
        return DM_ERR_INVALID_ARG;
    dm_shape_state* st = new (std::nothrow) dm_shape_state();
    if (!st) return DM_ERR_ALLOC;
    st->plan = p;
    st->prm = prm;
    const int n = p->n_vertices;
    st->n_blocks = (n + DM_SH_THREADS - 1) / DM_SH_THREADS;
    int rc = DM_OK;
    do {
        // the vertex graph: distinct neighbours of every vertex, ascending
        std::vector<int32_t> off, idx;
        try {
            std::vector<std::pair<int32_t, int32_t>> e;
            e.reserve((size_t)p->n_faces * 6);
            for (int32_t t = 0; t < p->n_faces; ++t)
                for (int a = 0; a < 3; ++a) {
                    const int32_t i = p->faces_host[3 * (size_t)t + a], j = p->faces_host[3 * (size_t)t + (a + 1) % 3];
                    if (i != j) {
                        e.emplace_back(i, j);
                        e.emplace_back(j, i);
                    }
                }
            std::sort(e.begin(), e.end());
            e.erase(std::unique(e.begin(), e.end()), e.end());
            off.assign((size_t)n + 1, 0);
            idx.resize(e.size());
            for (size_t q = 0; q < e.size(); ++q) {
                off[(size_t)e[q].first + 1]++;
                idx[q] = e[q].second;
            }
            int dmax = 0;
            for (int v = 0; v < n; ++v) {
                dmax = std::max(dmax, (int)off[(size_t)v + 1]);
                off[(size_t)v + 1] += off[v];
            }
            // CG on a symmetric positive definite matrix of condition number kappa reduces the A-norm of the error by
            // 2 ((sqrt(kappa)-1)/(sqrt(kappa)+1))^k; here 1 <= eig(I + lambda L) <= 1 + 2 lambda d_max (Gershgorin), so
            // k = 1/2 sqrt(kappa) ln(2 sqrt(kappa) / tol) iterations reach cg_tol in the 2-norm too: queue no more than
            // that (+ 10 %), the launches after convergence being no-ops that still cost their launch
            const double kap = 1.0 + 2.0 * (double)prm.lambda * (double)dmax;
            st->cg_iter_bound = (int)std::ceil(1.1 * 0.5 * std::sqrt(kap) * std::log(2.0 * std::sqrt(kap) / (double)prm.cg_tol)) + 2;
        } catch (...) { rc = DM_ERR_ALLOC; break; }
        const size_t n3 = (size_t)n * 3, nvox = (size_t)p->gd.nx * p->gd.ny * p->gd.nz, nb3 = (size_t)st->n_blocks * 3;
        if (cudaMalloc(&st->adj_off, off.size() * sizeof(int32_t)) != cudaSuccess ||
            cudaMalloc(&st->adj_idx, std::max<size_t>(1, idx.size()) * sizeof(int32_t)) != cudaSuccess ||
            cudaMalloc(&st->cg_x, n3 * sizeof(double)) != cudaSuccess || cudaMalloc(&st->cg_y, n3 * sizeof(double)) != cudaSuccess ||
            cudaMalloc(&st->cg_r, n3 * sizeof(double)) != cudaSuccess || cudaMalloc(&st->cg_p, n3 * sizeof(double)) != cudaSuccess ||
            cudaMalloc(&st->cg_Ap, n3 * sizeof(double)) != cudaSuccess || cudaMalloc(&st->part_a, nb3 * sizeof(double)) != cudaSuccess ||
            cudaMalloc(&st->part_b, nb3 * sizeof(double)) != cudaSuccess ||
            cudaMalloc(&st->cg_sc, 2 * sizeof(DmCgScalars)) != cudaSuccess || cudaMalloc(&st->cg_iters, 2 * sizeof(int)) != cudaSuccess || cudaMalloc(&st->cg_res, 2 * sizeof(double)) != cudaSuccess || cudaMalloc(&st->mom, n3 * sizeof(double)) != cudaSuccess ||
            cudaMalloc(&st->amax_part, DM_SH_LOSS_BLOCKS * sizeof(double)) != cudaSuccess ||
            cudaMalloc(&st->s_next, sizeof(double)) != cudaSuccess || cudaMalloc(&st->adam, sizeof(DmAdamScalars)) != cudaSuccess ||
            cudaMalloc(&st->image, nvox * sizeof(float)) != cudaSuccess || cudaMalloc(&st->cot, nvox * sizeof(float)) != cudaSuccess ||
            cudaMalloc(&st->grad, n3 * sizeof(float)) != cudaSuccess ||
            cudaMalloc(&st->loss_part, DM_SH_LOSS_BLOCKS * sizeof(double)) != cudaSuccess ||
            cudaMalloc(&st->loss, sizeof(double)) != cudaSuccess) { rc = DM_ERR_ALLOC; break; }
        if (cudaMemcpyAsync(st->adj_off, off.data(), off.size() * sizeof(int32_t), cudaMemcpyHostToDevice, p->stream) != cudaSuccess ||
            (!idx.empty() && cudaMemcpyAsync(st->adj_idx, idx.data(), idx.size() * sizeof(int32_t), cudaMemcpyHostToDevice, p->stream) !=
                                 cudaSuccess) ||
            cudaMemsetAsync(st->mom, 0, n3 * sizeof(double), p->stream) != cudaSuccess ||
            cudaMemsetAsync(st->adam, 0, sizeof(DmAdamScalars), p->stream) != cudaSuccess ||
            cudaMemsetAsync(st->cg_iters, 0, 2 * sizeof(int), p->stream) != cudaSuccess ||
            cudaMemsetAsync(st->cg_res, 0, 2 * sizeof(double), p->stream) != cudaSuccess ||
            cudaStreamSynchronize(p->stream) != cudaSuccess) { rc = DM_ERR_CUDA; break; }
        // the persistent solve needs every block resident at once (cooperative launch); blocks stride over the vertex tiles
        {
            int dev = 0, coop = 0, per_sm = 0;
            if (prm.solver == 0 && cudaGetDevice(&dev) == cudaSuccess && cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev) == cudaSuccess &&
                coop && cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, dm_k_cg_persistent<double>, DM_SH_THREADS, 0) == cudaSuccess &&
                per_sm > 0) {
                int per_sm_f = 0;
                cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm_f, dm_k_cg_persistent<float>, DM_SH_THREADS, 0);
                per_sm = std::min(per_sm, per_sm_f);
                // a vertex tile per block when they all fit; otherwise a grid that fills the machine once
                st->coop_blocks = std::min(st->n_blocks, per_sm * p->n_sm);
            }
            cudaGetLastError();
        }
    } while (0);
    if (rc != DM_OK) {
        dm_shape_state_destroy(st);
        cudaGetLastError();
        return rc;
    }
    *out = st;
    return DM_OK;
}

int dm_shape_precondition(dm_plan* p, dm_shape_state* st, const float* g_dev, float* out_dev)
{
    if (!p || !st || st->plan != p || !g_dev || !out_dev) return DM_ERR_INVALID_ARG;
    int rc = shape_precondition(p, st, g_dev);
    if (rc) return rc;
    const int n3 = p->n_vertices * 3;
    dm_k_f64_to_f32<<<(n3 + 255) / 256, 256, 0, p->stream>>>(st->cg_x, n3, out_dev);
    return check_launch(p);
}

int dm_shape_last_cg_iterations(dm_plan* p, dm_shape_state* st, int32_t iters[2])
{
    if (!p || !st || st->plan != p || !iters) return DM_ERR_INVALID_ARG;
    iters[0] = iters[1] = -1;
    if (st->coop_blocks <= 0) return DM_OK;   // the multi-launch solve keeps no count
    int h[2] = {0, 0};
    if (cudaMemcpyAsync(h, st->cg_iters, sizeof(h), cudaMemcpyDeviceToHost, p->stream) != cudaSuccess ||
        cudaStreamSynchronize(p->stream) != cudaSuccess)
        return DM_ERR_CUDA;
    iters[0] = h[0];
    iters[1] = h[1];
    return DM_OK;
}

int dm_shape_last_cg_residuals(dm_plan* p, dm_shape_state* st, double rel[2], int32_t* converged)
{
    if (!p || !st || st->plan != p || !rel) return DM_ERR_INVALID_ARG;
    if (cudaMemcpyAsync(rel, st->cg_res, 2 * sizeof(double), cudaMemcpyDeviceToHost, p->stream) != cudaSuccess ||
        cudaStreamSynchronize(p->stream) != cudaSuccess)
        return DM_ERR_CUDA;
    if (converged) *converged = (rel[0] <= (double)st->prm.cg_tol && rel[1] <= (double)st->prm.cg_tol) ? 1 : 0;
    return DM_OK;
}

int dm_shape_step(dm_plan* p, dm_shape_state* st, float* vertices_dev, const float* target_dev, const float* psf_cov_host,
                  double* loss_host)
{
    if (!p || !st || st->plan != p || !vertices_dev || !target_dev || !psf_cov_host) return DM_ERR_INVALID_ARG;
    int rc = dm_render(p, vertices_dev, psf_cov_host, st->image);
    if (rc) return rc;
    const long long nvox = (long long)p->gd.nx * p->gd.ny * p->gd.nz;
    dm_k_shape_loss<<<DM_SH_LOSS_BLOCKS, DM_SH_THREADS, 0, p->stream>>>(st->image, target_dev, nvox, st->cot, st->loss_part);
    dm_k_shape_loss_final<<<1, DM_SH_THREADS, 0, p->stream>>>(st->loss_part, DM_SH_LOSS_BLOCKS, st->loss);
    if ((rc = check_launch(p, 2))) return rc;
    // the vertices are the ones of the render above: its spectrum may be reused whatever DM_OPT_REUSE_SPECTRUM says
    const bool reuse_saved = p->reuse_F;
    p->reuse_F = true;
    rc = dm_render_backward(p, vertices_dev, psf_cov_host, st->cot, st->grad, nullptr);
    p->reuse_F = reuse_saved;
    if (rc) return rc;
    if ((rc = shape_precondition(p, st, st->grad))) return rc;
    const int n3 = p->n_vertices * 3;
    dm_k_adam_max<<<DM_SH_LOSS_BLOCKS, DM_SH_THREADS, 0, p->stream>>>(st->cg_x, n3, st->amax_part);
    dm_k_adam_update<<<(n3 + DM_SH_THREADS - 1) / DM_SH_THREADS, DM_SH_THREADS, 0, p->stream>>>(
        st->cg_x, n3, st->amax_part, DM_SH_LOSS_BLOCKS, st->mom, vertices_dev, st->adam, (double)st->prm.lr, (double)st->prm.beta1,
        (double)st->prm.beta2, (double)st->prm.eps, st->s_next);
    dm_k_adam_advance<<<1, 1, 0, p->stream>>>(st->adam, st->s_next);
    if ((rc = check_launch(p, 3))) return rc;
    p->F_valid = false;   // the vertices moved
    if (loss_host) {
        if (cudaMemcpyAsync(loss_host, st->loss, sizeof(double), cudaMemcpyDeviceToHost, p->stream) != cudaSuccess ||
            cudaStreamSynchronize(p->stream) != cudaSuccess)
            return DM_ERR_CUDA;
    }
    return DM_OK;
}

void dm_shape_state_destroy(dm_shape_state* st)
{
    if (!st) return;
    cudaFree(st->adj_off);
    cudaFree(st->adj_idx);
    cudaFree(st->cg_x);
    cudaFree(st->cg_y);
    cudaFree(st->cg_r);
    cudaFree(st->cg_p);
    cudaFree(st->cg_Ap);
    cudaFree(st->part_a);
    cudaFree(st->part_b);
    cudaFree(st->cg_sc);
    cudaFree(st->cg_iters);
    cudaFree(st->cg_res);
    cudaFree(st->mom);
    cudaFree(st->amax_part);
    cudaFree(st->s_next);
    cudaFree(st->adam);
    cudaFree(st->image);
    cudaFree(st->cot);
    cudaFree(st->grad);
    cudaFree(st->loss_part);
    cudaFree(st->loss);
    delete st;
}

}  // extern "C"

// ---- dm_mesh_ft_forward_noalloc: forward mesh FT for callers that must not allocate (include/deltamic.h) -----------------
//
// The plan-based forward keeps its scratch (triangle records, block sums of the k = 0 entry) in cudaMalloc'ed workspace.
// This variant keeps the same scratch in ONE array that is part of the library image: the driver places it in device
// memory when the module is loaded on a GPU and releases it when the process exits, so the call itself never asks the
// driver for memory.  Layout (bytes):  [0, 64 n_faces) triangle records of dm_k_geometry,
// [DM_NA_REC_BYTES, +8 DM_DC_BLOCKS) block sums of dm_k_dc_partial, then one double for dm_k_dc_final's total.
// All three regions are fully overwritten before they are read, so nothing has to start at zero.
namespace {

constexpr size_t DM_NA_REC_BYTES = (size_t)DM_NOALLOC_MAX_FACES * 4 * sizeof(float4);
constexpr size_t DM_NA_SCRATCH_BYTES = DM_NA_REC_BYTES + 1024;
static __device__ __align__(256) unsigned char dm_na_scratch[DM_NA_SCRATCH_BYTES];

// `dm_na_scratch` in HOST code is only a handle for the runtime, not a device address.  The address differs from GPU
// to GPU, so it is looked up once per device (with that device current) and remembered.
constexpr int DM_NA_MAX_DEVICES = 64;
void* g_na_ptr[DM_NA_MAX_DEVICES] = {};
std::mutex g_na_mutex;

int noalloc_scratch(unsigned char** out)
{
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= DM_NA_MAX_DEVICES) return DM_ERR_CUDA;
    std::lock_guard<std::mutex> lock(g_na_mutex);
    if (!g_na_ptr[dev]) {
        void* ptr = nullptr;
        if (cudaGetSymbolAddress(&ptr, dm_na_scratch) != cudaSuccess || !ptr) return DM_ERR_CUDA;
        g_na_ptr[dev] = ptr;
    }
    *out = static_cast<unsigned char*>(g_na_ptr[dev]);
    return DM_OK;
}

}  // namespace

extern "C" int dm_mesh_ft_forward_noalloc(const dm_grid* grid, int mode, const float* vertices_dev, const int32_t* faces_dev,
                                          int32_t n_faces, float* F_dev, void* cuda_stream)
{
    if (!grid || !vertices_dev || !faces_dev || !F_dev || n_faces <= 0 || (mode != DM_VOLUME && mode != DM_SURFACE))
        return DM_ERR_INVALID_ARG;
    for (int d = 0; d < 3; ++d)
        if (grid->n[d] <= 0 || grid->n[d] > 4096 || !(grid->spacing[d] > 0.f) || !std::isfinite(grid->spacing[d]))
            return DM_ERR_INVALID_ARG;
    if (grid->n[2] % 2 != 0) return DM_ERR_INVALID_ARG;
    if (n_faces > DM_NOALLOC_MAX_FACES) return DM_ERR_TOO_LARGE;   // the records would not fit the fixed array

    unsigned char* scratch = nullptr;
    int rc = noalloc_scratch(&scratch);   // first call on this device: looks the array's device address up
    if (rc) return rc;
    float4* rec = reinterpret_cast<float4*>(scratch);
    double* dc_part = reinterpret_cast<double*>(scratch + DM_NA_REC_BYTES);
    double* dc_total = dc_part + DM_DC_BLOCKS;

    DmGridDev gd;
    std::memset(&gd, 0, sizeof(gd));
    gd.nx = grid->n[0];
    gd.ny = grid->n[1];
    gd.nz = grid->n[2];
    gd.nzh = grid->n[2] / 2 + 1;
    double lmax = 0.0;
    for (int d = 0; d < 3; ++d) {
        const double L = (double)grid->n[d] * (double)grid->spacing[d];
        gd.kstep[d] = (float)(2.0 * M_PI / L);
        gd.inv_len[d] = 1.0 / L;
        lmax = std::max(lmax, L);
    }
    gd.band_lim = INFINITY;   // no narrow band, no face weights: the plain F of eq. 8-9
    gd.nzb = gd.nzh;
    gd.edge_fix = (float)(1073741824.0 / (lmax * lmax));
    gd.inv_edge_norm = (float)(1.0 / (3.0 * (double)n_faces * (double)gd.edge_fix));

    cudaStream_t stream = (cudaStream_t)cuda_stream;
    dm_k_geometry<<<(n_faces + 127) / 128, 128, 0, stream>>>(vertices_dev, faces_dev, n_faces, gd, rec);
    if (cudaGetLastError() != cudaSuccess) return DM_ERR_CUDA;
    const long long n_k = (long long)gd.nx * gd.ny * gd.nzh;
    dm_k_forward_robust<<<(unsigned)((n_k + 127) / 128), 128, 0, stream>>>(rec, n_faces, gd, mode, 0, gd.nx, (float2*)F_dev);
    if (cudaGetLastError() != cudaSuccess) return DM_ERR_CUDA;
    dm_k_dc_partial<<<DM_DC_BLOCKS, 256, 0, stream>>>(vertices_dev, faces_dev, n_faces, mode, nullptr, dc_part);
    if (cudaGetLastError() != cudaSuccess) return DM_ERR_CUDA;
    dm_k_dc_final<<<1, DM_DC_BLOCKS, 0, stream>>>(dc_part, F_dev, dc_total);
    return cudaGetLastError() == cudaSuccess ? DM_OK : DM_ERR_CUDA;
}
