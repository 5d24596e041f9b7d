// Prints the k-split decision of the backward mesh FT (paper_2303_10440_b200/csrc/dm_splits.h) for one problem size:
//   dump_splits n_x n_y n_zh n_faces n_sm band_on [ix_begin ix_end]   ->   "n_split_max n_split rows_per_split"
// Host-only; compiled with g++ by tests/test_host_topology.py.
#include <cstdio>
#include <cstdlib>

#include "../../paper_2303_10440_b200/csrc/dm_splits.h"

int main(int argc, char** argv)
{
    if (argc < 7) return 2;
    const int nx = atoi(argv[1]), ny = atoi(argv[2]), nzh = atoi(argv[3]);
    const long long n_faces = atoll(argv[4]);
    const int n_sm = atoi(argv[5]), band = atoi(argv[6]);
    const int ix0 = argc > 8 ? atoi(argv[7]) : 0, ix1 = argc > 8 ? atoi(argv[8]) : nx;
    const int split_target = 192, n_sums = 13;   // DM_BWD_SPLIT_TARGET, DM_BWD_NSUM of the library
    const int n_split_max = dm_backward_split_max(n_sm, split_target, n_sums, n_faces, (long long)nx * ny);
    int rps = 0;
    const int n_split = dm_backward_splits((ix1 - ix0) * ny, nzh, n_faces, n_sm, split_target, band != 0, n_split_max, &rps);
    printf("%d %d %d\n", n_split_max, n_split, rps);
    return 0;
}
