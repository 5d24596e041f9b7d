// dm_splits.h -- how the backward mesh FT divides the stored frequency rows (i_x, i_y) into k-splits.  Host arithmetic
// only (no CUDA), so that tests/host/dump_splits.cpp can check it without a GPU.
//
// One CTA of the backward kernels handles (one block of 128 triangles) x (one split of the rows).  The fast kernel
// (dm_k_backward_fast) stores a 15-bit row index inside the split in its queue entries, so a split may hold at most
// DM_SPLIT_MAX_ROWS rows; a launch that would need more falls back to the robust kernel (several times slower).
#pragma once
#include <algorithm>

#define DM_SPLIT_MAX_ROWS 32768

// Most splits a plan ever uses (sizes the partial-sum buffer [n_split_max][13][n_faces]): enough to fill the machine for a
// small mesh, within 64 M floats, and never fewer than the 15-bit row index needs on the whole grid.
inline int dm_backward_split_max(int n_sm, int split_target, int n_sums, long long n_faces, long long rows_whole_grid)
{
    const long long tri_blocks = (n_faces + 127) / 128;
    long long m = ((long long)n_sm * split_target + tri_blocks - 1) / tri_blocks;
    m = std::min<long long>(m, (64LL << 20) / ((long long)n_sums * n_faces));
    long long r = std::max<long long>(64, std::min<long long>(m, 4096));
    r = std::max<long long>(r, (rows_whole_grid + DM_SPLIT_MAX_ROWS - 1) / DM_SPLIT_MAX_ROWS);
    return (int)r;
}

// Splits of one launch over n_rows rows of n_zh stored frequencies each; *rows_per_split receives the rows of every split
// but the last.  With n_split_max from dm_backward_split_max, rows_per_split <= DM_SPLIT_MAX_ROWS always holds.
inline int dm_backward_splits(int n_rows, int n_zh, long long n_faces, int n_sm, int split_target, bool band_on,
                              int n_split_max, int* rows_per_split)
{
    // enough (triangle-block x k-split) CTAs to fill the machine (5 CTAs per SM) about 10 times over: short tail
    const long long tri_blocks = (n_faces + 127) / 128;
    long long want = ((long long)n_sm * split_target + tri_blocks - 1) / tri_blocks;
    if (band_on) want = std::max<long long>(want, std::min(n_split_max, 64));   // rows differ in cost under the narrow
                                                                                  // band: many small CTAs balance the load
    // a CTA sets up its seed table and records once: give it at least ~512 frequencies per triangle
    const int min_rows = (512 + n_zh - 1) / n_zh;
    if (want > n_rows / min_rows) want = n_rows / min_rows;
    if (want < 1) want = 1;
    // ... but never so few that a split outgrows the fast kernel's row index (large meshes on wide grids)
    want = std::max<long long>(want, ((long long)n_rows + DM_SPLIT_MAX_ROWS - 1) / DM_SPLIT_MAX_ROWS);
    if (want > n_rows) want = n_rows;
    if (want > n_split_max) want = n_split_max;
    const int rps = (int)((n_rows + want - 1) / want);
    *rows_per_split = rps;
    return (n_rows + rps - 1) / rps;
}
