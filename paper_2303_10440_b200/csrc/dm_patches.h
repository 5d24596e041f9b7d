// dm_patches.h -- host-side grouping of the mesh triangles into compact patches of 32 (built once per plan).
//
// The backward kernel (dm_bwd_fast.cuh) gives one WARP a patch of 32 triangles and lets the lanes share the vertex
// phases of the patch through shared memory: e^{-ik.v} kappa(k) is computed once per (frequency, patch vertex) and read
// by the (on average six) incident triangles of the patch (north_star: "each vertex's phase ... reused across its
// incident triangles").  A compact patch of 32 triangles has about 26 distinct vertices, so most warps compute ONE
// vertex phase per lane instead of three.  Topology only (faces), positions are not needed.
//
// Patches are grown as breadth-first balls over the face adjacency: a patch starts at the first unassigned face of a
// global breadth-first order, adds unassigned faces ring by ring until it holds 32, and -- when its ball runs out of
// unassigned faces first -- continues from the next unassigned face, so almost every patch holds exactly 32 faces.  A
// patch is closed early (its remaining lanes idle) when another face would push it past DM_PATCH_MAXV = 32 distinct
// vertices, one per lane: a few per cent of the patches, each losing a few lanes.
#pragma once
#include <cstdint>
#include <deque>
#include <vector>

#include "dm_strips.h"

#define DM_PATCH_FACES 32
#define DM_PATCH_MAXV 32   // vertex slots of a patch: lane l owns slot l

struct DmPatches {
    std::vector<int32_t> face;   // [n_patches*32]  face id of lane l, or -1 (idle lane)
    std::vector<int32_t> vid;    // [n_patches*32]  vertex id of slot s, or -1
    std::vector<uint32_t> loc;   // [n_patches*32]  slots of the face's corners 0,1,2: l0 | l1 << 8 | l2 << 16
    int64_t n_patches = 0;
};

inline DmPatches dm_build_patches(const int32_t* faces, int32_t n_f, int32_t n_v)
{
    using namespace dm_strips_detail;
    const Adj adj = build_adjacency(faces, n_f, n_v);
    auto for_neighbours = [&](int32_t f, auto&& fn) {
        for (int32_t q = adj.off[(size_t)3 * f]; q < adj.off[(size_t)3 * f + 3]; ++q) fn(adj.nbr[q]);
    };
    // global breadth-first order of the faces (component by component): the order in which patches are seeded
    std::vector<int32_t> order;
    order.reserve((size_t)n_f);
    {
        std::vector<char> seen((size_t)n_f, 0);
        for (int32_t s = 0; s < n_f; ++s) {
            if (seen[s]) continue;
            seen[s] = 1;
            size_t head = order.size();
            order.push_back(s);
            while (head < order.size()) {
                const int32_t f = order[head++];
                for_neighbours(f, [&](int32_t g) {
                    if (!seen[g]) {
                        seen[g] = 1;
                        order.push_back(g);
                    }
                });
            }
        }
    }
    DmPatches out;
    std::vector<char> assigned((size_t)n_f, 0);
    std::vector<int32_t> slot_of((size_t)n_v, -1);   // slot of a vertex in the CURRENT patch
    size_t seed_ptr = 0;
    int32_t n_assigned = 0;
    while (n_assigned < n_f) {
        std::vector<int32_t> pf, pv;
        std::deque<int32_t> q;
        while ((int)pf.size() < DM_PATCH_FACES) {
            if (q.empty()) {
                while (seed_ptr < order.size() && assigned[order[seed_ptr]]) ++seed_ptr;
                if (seed_ptr == order.size()) break;
                q.push_back(order[seed_ptr]);
            }
            const int32_t f = q.front();
            q.pop_front();
            if (assigned[f]) continue;
            int fresh = 0;
            for (int j = 0; j < 3; ++j) {
                const int32_t v = faces[3 * f + j];
                bool dup = false;
                for (int i = 0; i < j; ++i) dup = dup || faces[3 * f + i] == v;
                if (slot_of[v] < 0 && !dup) ++fresh;
            }
            if ((int)pv.size() + fresh > DM_PATCH_MAXV) break;   // close early (f stays unassigned)
            assigned[f] = 1;
            ++n_assigned;
            pf.push_back(f);
            for (int j = 0; j < 3; ++j) {
                const int32_t v = faces[3 * f + j];
                if (slot_of[v] < 0) {
                    slot_of[v] = (int32_t)pv.size();
                    pv.push_back(v);
                }
            }
            for_neighbours(f, [&](int32_t g) {
                if (!assigned[g]) q.push_back(g);
            });
        }
        // emit
        for (int l = 0; l < DM_PATCH_FACES; ++l) {
            if (l < (int)pf.size()) {
                const int32_t f = pf[l];
                out.face.push_back(f);
                out.loc.push_back((uint32_t)slot_of[faces[3 * f]] | ((uint32_t)slot_of[faces[3 * f + 1]] << 8) |
                                  ((uint32_t)slot_of[faces[3 * f + 2]] << 16));
            } else {
                out.face.push_back(-1);
                out.loc.push_back(0u);
            }
        }
        for (int s = 0; s < DM_PATCH_MAXV; ++s) out.vid.push_back(s < (int)pv.size() ? pv[s] : -1);
        for (int32_t v : pv) slot_of[v] = -1;
        ++out.n_patches;
    }
    return out;
}
