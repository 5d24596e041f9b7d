/*
 * deltamic.h -- C ABI of the B200-native (sm_100a) mesh Fourier transform of deltaMic
 * (arxiv 2303.10440, "Differentiable Rendering for 3D Fluorescence Microscopy").
 *
 * Citations are "PAPER.md:<line>" of the paper text plus the equation they fall in; "north_star" is
 * BASELINE.json's statement of the build.  Readings R1..R25 are listed in DESIGN.md section 3.
 *
 * The library renders a triangle mesh into a 3D image through the Fourier domain (Fig. 1,
 * :83-89 eq. 1-2):   image = irfft3( F . h_hat . e^{+i k.x0} ) / (h_x h_y h_z),
 * where F is the continuous Fourier transform of the mesh sampled on the image's rfft half-spectrum grid
 * (the hot path: dm_mesh_ft_forward / dm_mesh_ft_backward) and h_hat the spectrum of a Gaussian PSF
 * (eq. 3-4, reading R5).  Every step runs in CUDA kernels on one GPU; there is no CPU
 * fallback and no other backend.
 *
 * Conventions
 *  - Pointers named *_dev are DEVICE pointers owned by the caller (e.g. torch tensors' data_ptr());
 *    pointers named *_host are host pointers.  The plan owns its workspace and frees it in dm_plan_destroy.
 *  - Frequency grid (reading R10): spectrum arrays are [n_x][n_y][n_z/2+1], z fastest, complex64
 *    interleaved (re, im).  Index (i_x,i_y,i_z) holds integer frequency n_a = i_a for i_a < N_a/2,
 *    i_a - N_a otherwise (numpy fftfreq order) on x and y, n_z = i_z = 0..N_z/2; the angular frequency
 *    is k_a = 2 pi n_a / (N_a * spacing_a)  (PAPER.md:131 uses the angular convention e^{-i z.xi}).
 *  - Image arrays are [n_x][n_y][n_z] float32, z fastest.  Voxel (i,j,l) samples the point
 *    origin + (i h_x, j h_y, l h_z)  (readings R9, R11).
 *  - Vertices are float32 [n_vertices][3]; faces int32 [n_faces][3], counter-clockwise seen from outside
 *    (outward normal) -- a documented precondition of DM_VOLUME, not checked (reading R8).
 *  - Calls are asynchronous on the plan's CUDA stream unless stated.  Every call returns DM_OK (0) or a
 *    negative dm_status; nothing aborts, throws or prints.  Launch errors are returned by the call that
 *    made them, execution errors by the next call or the caller's own synchronisation.
 */
#ifndef DELTAMIC_H
#define DELTAMIC_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct dm_plan dm_plan; /* opaque */

typedef struct dm_grid {
    int32_t n[3];       /* voxels (x, y, z), 1..4096 each; the rfft half axis is z; n[2] must be even */
    float   spacing[3]; /* voxel size per axis; box length L_a = n[a] * spacing[a]             */
    float   origin[3];  /* sample point of voxel (0,0,0) (its centre), reading R11             */
} dm_grid;

typedef enum dm_mode {
    DM_VOLUME  = 0, /* F(k) = int_Omega e^{-ik.x} d^3x  (indicator of the enclosed volume; north_star)   */
    DM_SURFACE = 1  /* F(k) = sum_T int_T e^{-ik.x} dS  (membrane density; eq. 8-9,
                       :177-180 eq. 12 without the 1/|Lambda| normalisation, reading R7)                 */
} dm_mode;

typedef enum dm_status {
    DM_OK              =  0,
    DM_ERR_INVALID_ARG = -1, /* null pointer, non-positive size, odd n_z, unknown mode, bad slab        */
    DM_ERR_BAD_MESH    = -2, /* a face index is outside [0, n_vertices)                                 */
    DM_ERR_ALLOC       = -3, /* host or device allocation failed                                        */
    DM_ERR_CUDA        = -4, /* a CUDA runtime call or kernel launch failed                             */
    DM_ERR_CUFFT       = -5, /* a cuFFT call failed                                                     */
    DM_ERR_UNSUPPORTED = -6, /* the requested feature is not built                                      */
    DM_ERR_TOO_LARGE   = -7  /* dm_mesh_ft_forward_noalloc: n_faces > DM_NOALLOC_MAX_FACES                      */
} dm_status;

/* Create a plan for one grid, mode and mesh topology.
 *   faces_dev  device int32 [n_faces*3]; read (and validated) here and copied: the caller may free it
 *              afterwards.  A topology change needs a new plan; vertex positions may change freely.
 *   cuda_stream  a cudaStream_t (as void*); NULL = the legacy default stream.  All later calls on the
 *              plan are ordered on it.
 * This call synchronises the stream (it builds the vertex->corner CSR map of PAPER.md:182-186 eq. 13
 * and the cuFFT plans).  Returns DM_ERR_BAD_MESH for an out-of-range face index. */
int dm_plan_create(dm_plan** out, const dm_grid* grid, int mode, int32_t n_vertices, int32_t n_faces,
                   const int32_t* faces_dev, void* cuda_stream);

/* Move the plan to another CUDA stream: all later calls are ordered on it.  The caller orders the two streams (work already
 * queued on the old stream is not waited for).  Use: capture a whole optimisation step in a CUDA graph -- create the plan,
 * run every call of the step once (first calls allocate workspace, which cannot be captured), set the capturing stream,
 * capture, and replay; the 10 000-step fits of PAPER.md:261 on small meshes are launch-bound otherwise.  Inside a capture
 * nothing synchronises as long as dL_dpsf_cov_host / loss_host are NULL; dm_plan_stage_ms is meaningless for captured calls. */
int dm_plan_set_stream(dm_plan* plan, void* cuda_stream);

/* Restrict the mesh-FT calls of this plan to the x-slab [ix_begin, ix_end) of the stored spectrum
 * (array rows, not signed frequencies).  dm_mesh_ft_forward then writes only those rows of F and
 * dm_mesh_ft_backward sums only over them (a partial dL/dv that the caller all-reduces over slabs;
 * DESIGN.md section 9).  Default: the whole grid.  dm_render* require the whole grid. */
int dm_plan_set_slab(dm_plan* plan, int32_t ix_begin, int32_t ix_end);

/* Per-face density weights (the density is "a weighted sum" over surfaces of different fluorophore
 * concentration).  weights_dev = device float32 [n_faces], copied here (the caller may free it); every triangle term of
 * F, and so of the gradients, is multiplied by its face's weight: DM_SURFACE sum_T w_T int_T e^{-ik.x} dS, DM_VOLUME
 * (i/|k|^2) sum_T w_T (k.m_T) f_T (closed components with one weight each are regions of that density; negative weights
 * carve holes).  F(0) is the weighted area / volume.  NULL switches the weights off (all 1, the default).
 * Accuracy.  The tolerance of the unweighted path, max|dF| <= 1e-4 |F(0)|, carries over to weights
 * of ONE sign that, in DM_VOLUME, are constant on every connected component of the mesh (regions of different density):
 * those keep the fast kernels.  Any other weight set -- mixed signs (F(0) cancels and is no longer the scale of the
 * spectrum), or weights that vary inside a component in DM_VOLUME -- is evaluated pair by pair through the robust
 * series / far-pair branches (several times slower; dm_plan_paths_used reports it), and its tolerance is stated against
 * the scale of the same mesh with weights |w_T|:  max|dF| <= 1e-4 S_w,  S_w = sum_T |w_T| A_T  (DM_SURFACE)  or
 * sum_T |w_T| A_T L_max / (2 pi)  (DM_VOLUME; A_T L_max / (2 pi) bounds a triangle's term at the lowest non-zero
 * frequency).  The call reads the weights back to classify them, so it SYNCHRONISES the stream.  Non-finite weights
 * return DM_ERR_INVALID_ARG. */
int dm_plan_set_face_weights(dm_plan* plan, const float* weights_dev);

/* The same for a loop that refits the densities every step and cannot afford a stream
 * synchronisation and a host pass over the weights per step: copies weights_dev (device float32 [n_faces], not NULL)
 * asynchronously on the plan's stream and reads nothing back.  The caller states the class instead of having it
 * detected:  robust = 0 promises what dm_plan_set_face_weights checks for the fast kernels -- all weights finite and of
 * one sign and, in DM_VOLUME, equal on all faces of a connected component -- and robust = 1 sends every pair through
 * the robust kernels (always valid, several times slower).  A broken promise is not detected; the result may then miss
 * the tolerance.  Typical use: one dm_plan_set_face_weights call up front (allocates the plan's copy, classifies; read the
 * class back with dm_plan_paths_used after a forward), then this call inside the loop; once the plan's copy exists the
 * call allocates nothing and nothing in it synchronises. */
int dm_plan_update_face_weights(dm_plan* plan, const float* weights_dev, int32_t robust);

/* Narrow band ("evaluate the FT only where the PSF spectrum is above 1 % of its maximum").
 * With psf_cov_host = 6 floats on the HOST (covariance B of a Gaussian PSF, order xx, yy, zz, xy, xz, yz) and
 * 0 < cutoff < 1, the mesh-FT calls of this plan evaluate only the stored frequencies with
 * exp(-1/2 k^T B k) > cutoff: dm_mesh_ft_forward writes 0 everywhere else, dm_mesh_ft_backward ignores dL/dF there
 * (the gradient of the banded forward).  dm_render* use the band too; B is normally the PSF they are called with.
 * psf_cov_host = NULL switches the band off (the default).  k = 0 is always inside the band.  Setting the band
 * synchronises the stream (it builds the list of active frequencies).  A call that fails leaves the plan's previous
 * band (or no band) in force. */
int dm_plan_set_narrow_band(dm_plan* plan, const float* psf_cov_host, float cutoff);

/* Tuning / debugging knobs.  Defaults are the product path; the "robust" paths evaluate EVERY pair through the
 * series / far-pair branches (slow, used by the tests to cross-check the fast kernels at full size). */
typedef enum dm_option {
    DM_OPT_FORWARD_PATH  = 0, /* 0 = fast strip kernel (default), 1 = robust per-triangle kernel                  */
    DM_OPT_BACKWARD_PATH = 1, /* 0 = fast kernel (default), 1 = robust kernel                                     */
    DM_OPT_TAU           = 2, /* forward: gap-product threshold |pqr| at or below which a pair leaves the fast path (>= 0) */
    DM_OPT_TAU_BWD       = 3, /* backward: threshold on m1^2 m2 (the two smallest |gaps|) below which a pair leaves
                                 the fast path                                                                     */
    DM_OPT_AREA_NORMALISED = 4, /* DM_SURFACE only; 1 = the paper's membrane density u = F / |Lambda| (PAPER.md:177-186
                                  eq. 12) and its gradient (eq. 13): forward divides by the total area, backward takes
                                  dL/du and adds the -(sum_k Re(conj(G) u)/|Lambda|) d|Lambda|/dv term (it recomputes
                                  the forward once).  Whole grid only (a slab returns DM_ERR_UNSUPPORTED).  Default 0. */
    DM_OPT_REUSE_SPECTRUM = 5  /* 1 = the caller promises that every dm_render_backward is called with the vertices (and
                                  PSF mode) of the LAST dm_render on this plan, with no other forward call, setter or
                                  option change in between: the PSF-parameter gradient and eq. 13's extra term then take F
                                  from the spectrum dm_render left in the plan instead of recomputing the forward mesh FT
                                  (shape and PSF are fitted in the same loop).  The library cannot
                                  check the vertices; it returns DM_ERR_INVALID_ARG when the plan holds no such spectrum
                                  (no dm_render yet, or one of the calls above intervened).  Default 0 (recompute). */
} dm_option;
int dm_plan_set_option(dm_plan* plan, int option, double value);

/* Mesh Fourier transform (the hot path, forward).
 *   surface: F(k) = sum_T 2 A_T f_T(k),  f_T = eq. 9, evaluated through a numerically
 *            stable branch (series / divided differences) where the denominators of eq. 9 vanish or nearly
 *            vanish (eq. 14-16 done to full order, reading R4);
 *   volume:  F(k) = (i/|k|^2) sum_T (k.m_T) f_T(k),  m_T = (v2-v1)x(v3-v1),  F(0) = 1/6 sum_T v1.(v2 x v3).
 *   vertices_dev  float32 [n_vertices*3]
 *   F_dev         complex64 [n_x*n_y*(n_z/2+1)], overwritten (only the slab rows if a slab is set). */
int dm_mesh_ft_forward(dm_plan* plan, const float* vertices_dev, float* F_dev);

/* Vertex gradient of the mesh FT (the hot path, backward; PAPER.md:165-173 eq. 10-11, :182-186 eq. 13).
 *   dL_dF_dev  complex64, layout of F: G = dL/dRe F + i dL/dIm F for every STORED entry, all entries
 *              independent (reading R14).
 *   dL_dvertices_dev  float32 [n_vertices*3], overwritten with  sum_k Re( conj(G(k)) dF(k)/dv ).
 * Reduction over k per triangle is atomic-free and the scatter to vertices is a gather through the CSR
 * vertex->corner map, so results are bitwise reproducible run to run. */
int dm_mesh_ft_backward(dm_plan* plan, const float* vertices_dev, const float* dL_dF_dev,
                        float* dL_dvertices_dev);

/* dm_mesh_ft_backward for a caller that still holds the spectrum dm_mesh_ft_forward returned for THESE vertices
 * (F_dev, unchanged; the last forward call on the plan must have been that one): with DM_OPT_AREA_NORMALISED the
 * sum_k Re(conj(G) u) of eq. 13 is taken with it instead of a recomputed forward.  Without that option F_dev is unused
 * and the call equals dm_mesh_ft_backward. */
int dm_mesh_ft_backward_with_spectrum(dm_plan* plan, const float* vertices_dev, const float* dL_dF_dev,
                                      const float* F_dev, float* dL_dvertices_dev);

/* Whole forward render: mesh FT, multiply by the PSF spectrum and the origin shift, inverse real FFT.
 *   psf_cov_host  6 floats on the HOST: covariance of the Gaussian PSF in physical units, order
 *                 xx, yy, zz, xy, xz, yz;  h_hat(k) = exp(-1/2 k^T Sigma k)  (eq. 4 with reading R5).
 *   image_dev     float32 [n_x*n_y*n_z], overwritten. */
int dm_render(dm_plan* plan, const float* vertices_dev, const float* psf_cov_host, float* image_dev);

/* Backward of dm_render with respect to the vertices.
 *   dL_dimage_dev      float32 [n_x*n_y*n_z]
 *   dL_dvertices_dev   float32 [n_vertices*3], overwritten
 *   dL_dpsf_cov_host   NULL, or 6 floats on the HOST that receive dL/dSigma in the order of psf_cov_host
 *                      (the PSF parameters are fitted by gradient descent); an off-diagonal
 *                      entry is the derivative with respect to the one number that fills both symmetric positions.
 *                      When non-NULL the call needs the forward mesh FT of these vertices -- recomputed (one extra
 *                      dm_mesh_ft_forward) unless DM_OPT_REUSE_SPECTRUM is set -- and SYNCHRONISES the stream before
 *                      it returns (the six numbers land in host memory). */
int dm_render_backward(dm_plan* plan, const float* vertices_dev, const float* psf_cov_host,
                       const float* dL_dimage_dev, float* dL_dvertices_dev, float* dL_dpsf_cov_host);

/* The two surrounding stages on their own (used by the tests and the stage timing):
 *   dm_spectrum_to_image:  image = irfft3( F . h_hat . e^{+ik.x0} ) / (h_x h_y h_z)
 *   dm_image_to_spectrum_cotangent:  G = conj(h_hat e^{+ik.x0}) . w . rfft3(dL/dimage) / (N_tot h_x h_y h_z),
 *       w = 1 on the planes n_z = 0 and n_z = N_z/2, else 2 (the adjoint of the half-spectrum inverse
 *       transform on independent stored entries, reading R14).
 * F_dev is not modified. */
int dm_spectrum_to_image(dm_plan* plan, const float* F_dev, const float* psf_cov_host, float* image_dev);
int dm_image_to_spectrum_cotangent(dm_plan* plan, const float* dL_dimage_dev, const float* psf_cov_host,
                                   float* G_dev);

/* Device time of the stages of the LAST dm_render / dm_render_backward / dm_mesh_ft_* call, in ms:
 * ms[0] mesh FT (forward or backward reduction), ms[1] PSF multiply, ms[2] FFT, ms[3] scatter to
 * vertices.  Stages a call did not run report 0.  Synchronises the plan's stream. */
int dm_plan_stage_ms(dm_plan* plan, float ms[4]);

/* Number of CUDA kernels (cuFFT's excluded) the plan has launched since creation. */
int64_t dm_plan_launch_count(const dm_plan* plan);

/* Which kernels the LAST forward / backward mesh FT of this plan ran: paths[0] forward, paths[1] backward;
 * 0 = fast kernels, 1 = robust kernels (every pair through the series / far-pair branches: DM_OPT_*_PATH = 1, or a
 * weight set outside the fast kernels' validated regime), -1 = no such call yet.  Host-side bookkeeping, no sync.
 * (The fast backward kernel indexes the (i_x, i_y) rows of one k-split with 15 bits; the plan always cuts the grid into
 * enough splits for that -- csrc/dm_splits.h, at most 32768 rows each -- so grid or mesh size alone never selects the
 * robust kernel.) */
int dm_plan_paths_used(const dm_plan* plan, int32_t paths[2]);

void dm_plan_destroy(dm_plan* plan);

/* ---- Shape-optimisation step (section 5.1.3, eq. 17; readings R26-R28 of DESIGN.md) ------------------
 *   Phi_1 = sum_voxels (u - m)^2 m                      u = dm_render(vertices), m = the target image
 *   g     = dPhi_1/dvertices                            through dm_render_backward
 *   g~    = (I + lambda L)^-2 g                         L = D - A, the connectivity Laplacian of the mesh's vertex graph;
 *                                                       two conjugate-gradient solves with I + lambda L on the device
 *                                                       (the paper uses a sparse Cholesky factorisation), fp64; one
 *                                                       persistent cooperative kernel per solve wherever the device
 *                                                       supports cooperative launches (its blocks stride over the vertex
 *                                                       tiles when the mesh has more tiles than one resident grid,
 *                                                       ~3e5 vertices), else three launches per iteration
 *   vertices <- AdamUniform(vertices, g~)               m_t = b1 m + (1-b1) g~,  s_t = b2 s + (1-b2) max_i g~_i^2,
 *                                                       v -= lr (m_t/(1-b1^t)) / (sqrt(s_t/(1-b2^t)) + eps)
 * The state owns the vertex graph, the optimiser moments (zero at creation) and all scratch; it belongs to ONE plan
 * (and must be destroyed before it).  The step honours the plan's narrow band (the shape step runs on
 * the narrow band), slab must be the whole grid.  Everything is queued on the plan's stream; nothing synchronises
 * unless loss_host is given. */
typedef struct dm_shape_state dm_shape_state; /* opaque */

typedef struct dm_shape_params {
    float   lr;          /* eta of eq. 17 (default 1e-3)                                              */
    float   lambda;      /* diffusion weight (default 50)                               */
    float   beta1;       /* first-moment decay (default 0.9)                                          */
    float   beta2;       /* second-moment decay (default 0.999)                                       */
    float   eps;         /* default 1e-8                                                              */
    float   cg_tol;      /* a solve stops when |r| <= cg_tol |b| on every column (default 1e-7)       */
    int32_t cg_max_iter; /* at most this many iterations are queued per solve (default 400); fewer when
                            the convergence bound of CG for cond(I + lambda L) <= 1 + 2 lambda d_max says so */
    int32_t solver;      /* 0 = automatic (default): one persistent cooperative kernel per solve whenever the device
                            supports cooperative launches (a refused launch falls back to 1);  1 = three launches per
                            iteration.  Same arithmetic; the results agree bit for bit while every 256-vertex tile has a
                            block of its own in the resident grid (~3e5 vertices on a B200) -- beyond that the persistent
                            solve sums its dot products in a different order and the two differ by rounding */
} dm_shape_params;

int dm_shape_params_default(dm_shape_params* out);

/* params = NULL takes the defaults.  Synchronises the stream (it uploads the vertex graph). */
int dm_shape_state_create(dm_plan* plan, const dm_shape_params* params, dm_shape_state** out);

/* out = (I + lambda L)^-2 g for a float32 [n_vertices*3] field g (both DEVICE pointers; they may be the same). */
int dm_shape_precondition(dm_plan* plan, dm_shape_state* state, const float* g_dev, float* out_dev);

/* Conjugate-gradient iterations the two solves of the last dm_shape_precondition / dm_shape_step took (iters[0], iters[1]);
 * -1 when the solves ran as separate launches (solver = 1, or a refused cooperative launch), which keep no count.
 * Synchronises the stream. */
int dm_shape_last_cg_iterations(dm_plan* plan, dm_shape_state* state, int32_t iters[2]);

/* How well those two solves converged: rel[i] = max over the three columns of |r| / |b| when solve i stopped (0 before
 * any solve).  Both solver forms stop silently after cg_max_iter iterations (a large lambda needs more: the iteration
 * count grows like sqrt(1 + 2 lambda d_max)); *converged (may be NULL) is 1 when both rel[i] <= cg_tol, 0 when a solve
 * ran out of iterations first -- the step was then taken with an inexactly preconditioned gradient.  Synchronises the
 * stream. */
int dm_shape_last_cg_residuals(dm_plan* plan, dm_shape_state* state, double rel[2], int32_t* converged);

/* One step.  vertices_dev float32 [n_vertices*3] is updated IN PLACE; target_dev float32 [n_x*n_y*n_z] is the image m;
 * psf_cov_host as in dm_render.  loss_host = NULL, or a HOST double that receives Phi_1 of the vertices BEFORE the
 * step (the call then synchronises the stream). */
int dm_shape_step(dm_plan* plan, dm_shape_state* state, float* vertices_dev, const float* target_dev,
                  const float* psf_cov_host, double* loss_host);

void dm_shape_state_destroy(dm_shape_state* state);

/* ---- Forward mesh FT without a plan and without any memory allocation ----------------------------------------------------
 * Who this is for.  Everything above goes through a plan, and a plan gets its workspace from cudaMalloc (at creation, and
 * lazily on some first calls).  Some programs cannot afford that: a process that gave the whole GPU to one arena at start-up
 * (a framework's caching allocator, a fixed memory budget per service) may find that a raw cudaMalloc fails or is forbidden
 * by policy; a latency-bound loop cannot accept that cudaMalloc / cudaFree stall the device while they run; and code called
 * from inside someone else's pipeline often has no say over when allocation is allowed.  Such callers hand in their own
 * input and output buffers and call this function, which asks the CUDA runtime for no memory at all (no cudaMalloc, no
 * cudaFree, no cuFFT or other allocating library routine, no host allocation).
 *
 * What it computes.  The same F as dm_mesh_ft_forward on a fresh plan of this grid and mode (whole grid, no narrow band, no
 * face weights, no area normalisation; eq. 8-9, volume mode as above), with every (triangle, frequency)
 * pair evaluated through the series / far-pair branches -- the kernels a plan runs under DM_OPT_FORWARD_PATH = 1.  It meets
 * the same tolerance (max|dF| <= 1e-4 |F(0)|) but is several times slower than the plan's strip kernel: it is meant for
 * small and medium meshes, not for the bench workloads.
 *
 * Where the scratch lives.  The triangle records (64 bytes per face) and the block sums of the k = 0 entry sit in a
 * fixed array compiled into the library, DM_NOALLOC_MAX_FACES * 64 + 1024 bytes (4 MiB + 1 KiB).  Every GPU on which the
 * library's kernels are loaded carries that array until the process exits, whether or not this function is ever called.
 * n_faces > DM_NOALLOC_MAX_FACES returns DM_ERR_TOO_LARGE before anything is launched.
 *
 * Sharing.  There is one array per GPU and every call on that GPU uses it, from any thread and on any stream.  Two calls
 * whose kernels can run at the same time on one GPU (different streams without an event between them, or two host
 * threads) overwrite each other's records and both results are garbage: the caller serialises them.  Calls on one stream,
 * or on different GPUs, are safe.  The array keeps whatever the previous call left in it; this function overwrites every
 * byte it later reads, so no clearing is needed and a call never sees an earlier call's data.
 *
 * First call on a GPU.  The first call made while a given device is current looks up that device's address of the array
 * (cudaGetSymbolAddress; this may also make the runtime load the library's kernels onto that GPU) and remembers it.  Make
 * that first call during set-up, with the device you will use current, before any CUDA stream capture is begun.
 *
 *   grid          as in dm_plan_create (origin is not used by the mesh FT)
 *   vertices_dev  device float32 [n_vertices*3]
 *   faces_dev     device int32 [n_faces*3]; indices must lie inside the vertex array -- NOT checked here (checking needs a
 *                 copy to the host), an out-of-range index reads out of bounds
 *   F_dev         device complex64 [n_x*n_y*(n_z/2+1)], overwritten
 *   cuda_stream   a cudaStream_t; NULL = the legacy default stream.  The call is asynchronous on it.
 * Returns DM_OK, DM_ERR_INVALID_ARG, DM_ERR_TOO_LARGE or DM_ERR_CUDA. */
#define DM_NOALLOC_MAX_FACES 65536
int dm_mesh_ft_forward_noalloc(const dm_grid* grid, int mode, const float* vertices_dev, const int32_t* faces_dev,
                               int32_t n_faces, float* F_dev, void* cuda_stream);

const char* dm_error_string(int code);

/* Library version as major*10000 + minor*100 + patch. */
int dm_version(void);

#ifdef __cplusplus
}
#endif
#endif /* DELTAMIC_H */
