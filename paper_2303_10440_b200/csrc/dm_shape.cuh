// dm_shape.cuh -- kernels of the shape-optimisation step (section 5.1.3, eq. 17), sm_100a.
//
//   Phi_1 = sum_voxels (u - m)^2 m                       (kappa = 1)
//   v <- v - eta (I + lambda L)^-2 dPhi_1/dv             (eq. 17), stepped by AdamUniform (ref. [55])
//
// L = D - A is the connectivity Laplacian of the mesh's vertex graph (reading R26), kept as a CSR list of the distinct
// neighbours of every vertex.  The paper factorises I + lambda L with a sparse Cholesky decomposition on the host; here
// the two solves with M = I + lambda L (reading R27) are conjugate-gradient solves that never leave the device: M is
// symmetric positive definite with condition number <= 1 + 2 lambda max_degree (about 700 for lambda = 50), the three
// coordinate columns are solved at once with their own step lengths, vectors and dot products are fp64 (the work is
// O(n_V) per iteration, nothing next to the mesh FT), and every reduction is a fixed-order two-stage tree, so the step is
// bitwise reproducible.  The solve is one persistent cooperative kernel (three grid barriers per iteration, it stops at
// convergence) when every block fits on the device at once, else three small launches per iteration with a device flag that
// turns the launches of a converged solve into no-ops; either way the host never synchronises.
// AdamUniform (reading R28): Adam whose second moment is one scalar per step, the largest squared gradient entry.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#define DM_SH_THREADS 256
#define DM_SH_LOSS_BLOCKS 256

// fixed-order block sum of one double per thread (DM_SH_THREADS threads); every thread gets the result
__device__ __forceinline__ double dm_sh_block_sum(double v, double* sh)
{
    __syncthreads();
    sh[threadIdx.x] = v;
    __syncthreads();
    for (int s = DM_SH_THREADS / 2; s > 0; s >>= 1) {
        if ((int)threadIdx.x < s) sh[threadIdx.x] += sh[threadIdx.x + s];
        __syncthreads();
    }
    return sh[0];
}
__device__ __forceinline__ double dm_sh_block_max(double v, double* sh)
{
    __syncthreads();
    sh[threadIdx.x] = v;
    __syncthreads();
    for (int s = DM_SH_THREADS / 2; s > 0; s >>= 1) {
        if ((int)threadIdx.x < s) sh[threadIdx.x] = fmax(sh[threadIdx.x], sh[threadIdx.x + s]);
        __syncthreads();
    }
    return sh[0];
}
// the total of n_part block partials [n_part][3], computed by every block alike (thread-strided, then the block tree)
__device__ __forceinline__ void dm_sh_total3(const double* __restrict__ part, int n_part, double* sh, double out[3])
{
    for (int c = 0; c < 3; ++c) {
        double a = 0.0;
        for (int i = threadIdx.x; i < n_part; i += DM_SH_THREADS) a += part[3 * (size_t)i + c];
        out[c] = dm_sh_block_sum(a, sh);
    }
}

// ---- Phi_1 and its image cotangent -------------------------------------------------------------------------------------
//   cot = dPhi_1/du = 2 (u - m) m ;  partial[b] = block sums of (u - m)^2 m   (fp64)
__global__ void __launch_bounds__(DM_SH_THREADS)
dm_k_shape_loss(const float* __restrict__ u, const float* __restrict__ m, long long n, float* __restrict__ cot,
                double* __restrict__ partial)
{
    __shared__ double sh[DM_SH_THREADS];
    double acc = 0.0;
    for (long long l = (long long)blockIdx.x * blockDim.x + threadIdx.x; l < n; l += (long long)gridDim.x * blockDim.x) {
        const float d = u[l] - m[l], w = m[l];
        cot[l] = 2.0f * d * w;
        acc += (double)d * (double)d * (double)w;
    }
    const double s = dm_sh_block_sum(acc, sh);
    if (threadIdx.x == 0) partial[blockIdx.x] = s;
}
__global__ void __launch_bounds__(DM_SH_THREADS)
dm_k_shape_loss_final(const double* __restrict__ partial, int n_part, double* __restrict__ loss)
{
    __shared__ double sh[DM_SH_THREADS];
    double a = 0.0;
    for (int i = threadIdx.x; i < n_part; i += DM_SH_THREADS) a += partial[i];
    const double s = dm_sh_block_sum(a, sh);
    if (threadIdx.x == 0) *loss = s;
}

// ---- conjugate gradients on M = I + lambda L, three right-hand sides at once -------------------------------------------
struct DmCgScalars {
    double rr[3];   // r.r of every column
    double bb[3];   // b.b of every column (the convergence scale)
    int done;       // every column has r.r <= tol^2 b.b
};

// max over the three columns of |r| / |b| (0 for a zero right-hand side)
__device__ __forceinline__ double dm_sh_rel_residual(const double rr[3], const double bb[3])
{
    double m = 0.0;
    for (int c = 0; c < 3; ++c)
        if (bb[c] > 0.0) m = fmax(m, sqrt(rr[c] / bb[c]));
    return m;
}

// x = 0, r = p = b (b given as fp32 [n][3] or fp64), partial r.r
template <typename TB>
__global__ void __launch_bounds__(DM_SH_THREADS)
dm_k_cg_init(const TB* __restrict__ b, int n, double* __restrict__ x, double* __restrict__ r, double* __restrict__ p,
             double* __restrict__ part)
{
    __shared__ double sh[DM_SH_THREADS];
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    double v[3] = {0.0, 0.0, 0.0};
    if (i < n)
        for (int c = 0; c < 3; ++c) {
            v[c] = (double)b[3 * (size_t)i + c];
            x[3 * (size_t)i + c] = 0.0;
            r[3 * (size_t)i + c] = v[c];
            p[3 * (size_t)i + c] = v[c];
        }
    for (int c = 0; c < 3; ++c) {
        const double s = dm_sh_block_sum(v[c] * v[c], sh);
        if (threadIdx.x == 0) part[3 * (size_t)blockIdx.x + c] = s;
    }
}
__global__ void __launch_bounds__(DM_SH_THREADS)
dm_k_cg_init_final(const double* __restrict__ part, int n_part, DmCgScalars* __restrict__ sc)
{
    __shared__ double sh[DM_SH_THREADS];
    double t[3];
    dm_sh_total3(part, n_part, sh, t);
    if (threadIdx.x == 0) {
        for (int c = 0; c < 3; ++c) sc->rr[c] = sc->bb[c] = t[c];
        sc->done = (t[0] == 0.0 && t[1] == 0.0 && t[2] == 0.0) ? 1 : 0;
    }
}
// Ap = p + lambda (deg p - sum_neighbours p), partial p.Ap
__global__ void __launch_bounds__(DM_SH_THREADS)
dm_k_cg_spmv(const int32_t* __restrict__ adj_off, const int32_t* __restrict__ adj_idx, int n, double lambda,
             const double* __restrict__ p, double* __restrict__ Ap, double* __restrict__ part,
             const DmCgScalars* __restrict__ sc)
{
    __shared__ double sh[DM_SH_THREADS];
    if (sc->done) return;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    double d[3] = {0.0, 0.0, 0.0};
    if (i < n) {
        const int b = adj_off[i], e = adj_off[i + 1];
        double s[3] = {0.0, 0.0, 0.0};
        for (int j = b; j < e; ++j) {
            const size_t q = 3 * (size_t)adj_idx[j];
            s[0] += p[q], s[1] += p[q + 1], s[2] += p[q + 2];
        }
        const double deg = (double)(e - b);
        for (int c = 0; c < 3; ++c) {
            const double pi = p[3 * (size_t)i + c];
            const double a = pi + lambda * (deg * pi - s[c]);
            Ap[3 * (size_t)i + c] = a;
            d[c] = pi * a;
        }
    }
    for (int c = 0; c < 3; ++c) {
        const double s = dm_sh_block_sum(d[c], sh);
        if (threadIdx.x == 0) part[3 * (size_t)blockIdx.x + c] = s;
    }
}
// alpha = r.r / p.Ap ; x += alpha p ; r -= alpha Ap ; partial of the new r.r
__global__ void __launch_bounds__(DM_SH_THREADS)
dm_k_cg_update_x(int n, const double* __restrict__ p, const double* __restrict__ Ap, double* __restrict__ x,
                 double* __restrict__ r, const double* __restrict__ part_pAp, double* __restrict__ part_rr, int n_part,
                 const DmCgScalars* __restrict__ sc)
{
    __shared__ double sh[DM_SH_THREADS];
    if (sc->done) return;
    double pAp[3];
    dm_sh_total3(part_pAp, n_part, sh, pAp);
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    double d[3] = {0.0, 0.0, 0.0};
    if (i < n)
        for (int c = 0; c < 3; ++c) {
            const double alpha = pAp[c] > 0.0 ? sc->rr[c] / pAp[c] : 0.0;   // a column that has converged exactly stays put
            const size_t q = 3 * (size_t)i + c;
            x[q] += alpha * p[q];
            const double rn = r[q] - alpha * Ap[q];
            r[q] = rn;
            d[c] = rn * rn;
        }
    for (int c = 0; c < 3; ++c) {
        const double s = dm_sh_block_sum(d[c], sh);
        if (threadIdx.x == 0) part_rr[3 * (size_t)blockIdx.x + c] = s;
    }
}
// beta = r.r(new) / r.r(old) ; p = r + beta p ; block 0 writes the scalars of the NEXT iteration into the other buffer
// (sc_next != sc: every block may still be reading sc): the new r.r and the convergence test r.r <= tol^2 b.b on every column
__global__ void __launch_bounds__(DM_SH_THREADS)
dm_k_cg_update_p(int n, const double* __restrict__ r, double* __restrict__ p, const double* __restrict__ part_rr,
                 int n_part, const DmCgScalars* __restrict__ sc, DmCgScalars* __restrict__ sc_next, double tol2)
{
    __shared__ double sh[DM_SH_THREADS];
    if (sc->done) {
        if (blockIdx.x == 0 && threadIdx.x == 0) *sc_next = *sc;
        return;
    }
    double rn[3];
    dm_sh_total3(part_rr, n_part, sh, rn);
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n)
        for (int c = 0; c < 3; ++c) {
            const double beta = sc->rr[c] > 0.0 ? rn[c] / sc->rr[c] : 0.0;
            const size_t q = 3 * (size_t)i + c;
            p[q] = r[q] + beta * p[q];
        }
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        bool all = true;
        for (int c = 0; c < 3; ++c) {
            sc_next->rr[c] = rn[c];
            sc_next->bb[c] = sc->bb[c];
            all = all && (rn[c] <= tol2 * sc->bb[c]);
        }
        sc_next->done = all ? 1 : 0;
    }
}

// ---- AdamUniform (reading R28) -------------------------------------------------------------------------------------------
struct DmAdamScalars {
    double s;   // scalar second moment
    int t;      // steps taken
};
__global__ void __launch_bounds__(DM_SH_THREADS)
dm_k_adam_max(const double* __restrict__ g, int n3, double* __restrict__ part)
{
    __shared__ double sh[DM_SH_THREADS];
    double a = 0.0;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n3; i += gridDim.x * blockDim.x) a = fmax(a, g[i] * g[i]);
    const double m = dm_sh_block_max(a, sh);
    if (threadIdx.x == 0) part[blockIdx.x] = m;
}
//   m = b1 m + (1 - b1) g ;  s = b2 s + (1 - b2) max g^2 ;  v -= lr (m / (1 - b1^t)) / (sqrt(s / (1 - b2^t)) + eps)
// sc is read here and advanced by dm_k_adam_advance afterwards.
__global__ void __launch_bounds__(DM_SH_THREADS)
dm_k_adam_update(const double* __restrict__ g, int n3, const double* __restrict__ part, int n_part, double* __restrict__ mom,
                 float* __restrict__ vertices, const DmAdamScalars* __restrict__ sc, double lr, double b1, double b2, double eps,
                 double* __restrict__ s_next)
{
    __shared__ double sh[DM_SH_THREADS];
    double a = 0.0;
    for (int i = threadIdx.x; i < n_part; i += DM_SH_THREADS) a = fmax(a, part[i]);
    const double gmax2 = dm_sh_block_max(a, sh);
    const int t = sc->t + 1;
    const double s = b2 * sc->s + (1.0 - b2) * gmax2;
    const double c1 = 1.0 - pow(b1, (double)t), c2 = 1.0 - pow(b2, (double)t);
    const double denom = sqrt(s / c2) + eps;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n3) {
        const double m = b1 * mom[i] + (1.0 - b1) * g[i];
        mom[i] = m;
        vertices[i] = (float)((double)vertices[i] - lr * (m / c1) / denom);
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) *s_next = s;
}
__global__ void dm_k_adam_advance(DmAdamScalars* __restrict__ sc, const double* __restrict__ s_next)
{
    sc->s = *s_next;
    sc->t += 1;
}

__global__ void dm_k_f64_to_f32(const double* __restrict__ a, int n, float* __restrict__ out)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) out[i] = (float)a[i];
}

// ---- the same conjugate-gradient solve as ONE persistent kernel (cooperative launch, grid-wide barriers) ----------------
// Used when every block of the solve can be resident at once (always, up to ~3e5 vertices): the three launches per iteration
// become three grid barriers, and the kernel STOPS at convergence instead of queueing no-op launches.  The arithmetic and
// the order of every sum are those of the multi-launch kernels above (block partials in block order, every block adds them
// alike), with the vertices of a block being the tiles blockIdx.x, blockIdx.x + gridDim.x, ...
#include <cooperative_groups.h>

// fixed-order block sum of three doubles per thread; every thread gets the results
__device__ __forceinline__ void dm_sh_block_sum3(double v[3], double (*sh)[DM_SH_THREADS])
{
    __syncthreads();
#pragma unroll
    for (int c = 0; c < 3; ++c) sh[c][threadIdx.x] = v[c];
    __syncthreads();
    for (int s = DM_SH_THREADS / 2; s > 0; s >>= 1) {
        if ((int)threadIdx.x < s)
#pragma unroll
            for (int c = 0; c < 3; ++c) sh[c][threadIdx.x] += sh[c][threadIdx.x + s];
        __syncthreads();
    }
#pragma unroll
    for (int c = 0; c < 3; ++c) v[c] = sh[c][0];
}
// block partials out, grid barrier, total of all blocks' partials (the same on every block)
__device__ __forceinline__ void dm_sh_grid_sum3(double v[3], double* __restrict__ part, double (*sh)[DM_SH_THREADS])
{
    dm_sh_block_sum3(v, sh);
    if (threadIdx.x == 0)
#pragma unroll
        for (int c = 0; c < 3; ++c) part[3 * (size_t)blockIdx.x + c] = v[c];
    cooperative_groups::this_grid().sync();
    double a[3] = {0.0, 0.0, 0.0};
    for (int i = threadIdx.x; i < (int)gridDim.x; i += DM_SH_THREADS)
#pragma unroll
        for (int c = 0; c < 3; ++c) a[c] += part[3 * (size_t)i + c];
    dm_sh_block_sum3(a, sh);
#pragma unroll
    for (int c = 0; c < 3; ++c) v[c] = a[c];
}

template <typename TB>
__global__ void __launch_bounds__(DM_SH_THREADS)
dm_k_cg_persistent(const int32_t* __restrict__ adj_off, const int32_t* __restrict__ adj_idx, int n, double lambda,
                   const TB* __restrict__ b, double* __restrict__ x, double* __restrict__ r, double* __restrict__ p,
                   double* __restrict__ Ap, double* __restrict__ part_a, double* __restrict__ part_b, double tol2, int max_iter,
                   int* __restrict__ iters_out, double* __restrict__ res_out)
{
    __shared__ double sh[3][DM_SH_THREADS];
    const int stride = (int)gridDim.x * DM_SH_THREADS;
    const int i0 = (int)blockIdx.x * DM_SH_THREADS + (int)threadIdx.x;
    double rr[3] = {0.0, 0.0, 0.0}, bb[3];
    for (int i = i0; i < n; i += stride)
        for (int c = 0; c < 3; ++c) {
            const double v = (double)b[3 * (size_t)i + c];
            x[3 * (size_t)i + c] = 0.0;
            r[3 * (size_t)i + c] = v;
            p[3 * (size_t)i + c] = v;
            rr[c] += v * v;
        }
    dm_sh_grid_sum3(rr, part_a, sh);
    for (int c = 0; c < 3; ++c) bb[c] = rr[c];
    int it = 0;
    for (; it < max_iter; ++it) {
        if (rr[0] <= tol2 * bb[0] && rr[1] <= tol2 * bb[1] && rr[2] <= tol2 * bb[2]) break;   // the same on every block
        double pAp[3] = {0.0, 0.0, 0.0};
        for (int i = i0; i < n; i += stride) {
            const int jb = adj_off[i], je = adj_off[i + 1];
            double s[3] = {0.0, 0.0, 0.0};
            for (int j = jb; j < je; ++j) {
                const size_t q = 3 * (size_t)adj_idx[j];
                s[0] += p[q], s[1] += p[q + 1], s[2] += p[q + 2];
            }
            const double deg = (double)(je - jb);
            for (int c = 0; c < 3; ++c) {
                const double pi = p[3 * (size_t)i + c];
                const double a = pi + lambda * (deg * pi - s[c]);
                Ap[3 * (size_t)i + c] = a;
                pAp[c] += pi * a;
            }
        }
        dm_sh_grid_sum3(pAp, part_b, sh);
        double rn[3] = {0.0, 0.0, 0.0};
        for (int i = i0; i < n; i += stride)
            for (int c = 0; c < 3; ++c) {
                const double alpha = pAp[c] > 0.0 ? rr[c] / pAp[c] : 0.0;
                const size_t q = 3 * (size_t)i + c;
                x[q] += alpha * p[q];
                const double rv = r[q] - alpha * Ap[q];
                r[q] = rv;
                rn[c] += rv * rv;
            }
        dm_sh_grid_sum3(rn, part_a, sh);
        for (int i = i0; i < n; i += stride)
            for (int c = 0; c < 3; ++c) {
                const double beta = rr[c] > 0.0 ? rn[c] / rr[c] : 0.0;
                const size_t q = 3 * (size_t)i + c;
                p[q] = r[q] + beta * p[q];
            }
        for (int c = 0; c < 3; ++c) rr[c] = rn[c];
        cooperative_groups::this_grid().sync();   // p is complete before the next product reads the neighbours
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        if (iters_out) *iters_out = it;
        if (res_out) *res_out = dm_sh_rel_residual(rr, bb);
    }
}

// the relative residual the multi-launch solve ended with (its scalars live in sc)
__global__ void dm_k_cg_residual(const DmCgScalars* __restrict__ sc, double* __restrict__ res_out)
{
    *res_out = dm_sh_rel_residual(sc->rr, sc->bb);
}
