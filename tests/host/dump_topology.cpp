// Test harness for the host-side topology builders of the CUDA library (dm_strips.h, dm_patches.h): reads a face list,
// writes the strip records and the patches as text for tests/test_host_topology.py.  Host C++ only, no CUDA.
#include <cstdio>
#include <vector>

#include "../../paper_2303_10440_b200/csrc/dm_patches.h"

int main(int argc, char** argv)
{
    if (argc < 3) return 2;
    FILE* f = fopen(argv[1], "rb");
    if (!f) return 3;
    int32_t nf = 0, nv = 0;
    if (fread(&nf, 4, 1, f) != 1 || fread(&nv, 4, 1, f) != 1) return 4;
    std::vector<int32_t> F(3 * (size_t)nf);
    if (fread(F.data(), 4, F.size(), f) != F.size()) return 5;
    fclose(f);
    const int n_chunks = argc > 3 ? atoi(argv[3]) : 4;
    const DmPatches p = dm_build_patches(F.data(), nf, nv);
    const DmStripRecords s = dm_build_strips(F.data(), nf, nv, n_chunks);
    FILE* o = fopen(argv[2], "w");
    if (!o) return 6;
    fprintf(o, "patches %lld\n", (long long)p.n_patches);
    for (size_t i = 0; i < p.face.size(); ++i) fprintf(o, "%d %d %u\n", p.face[i], p.vid[i], p.loc[i]);
    fprintf(o, "strips %lld records %zu chunks %zu\n", (long long)s.n_strips, s.fid.size(), s.chunk_off.size() - 1);
    for (size_t c = 0; c < s.chunk_off.size(); ++c) fprintf(o, "%d\n", s.chunk_off[c]);
    for (size_t i = 0; i < s.fid.size(); ++i) fprintf(o, "%d %d %d %d\n", s.vid_new[i], s.vid_prev[i], s.vid_ret[i], s.fid[i]);
    fclose(o);
    return 0;
}
