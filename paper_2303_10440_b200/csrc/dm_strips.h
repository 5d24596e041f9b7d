// dm_strips.h -- host-side triangle-strip decomposition of the mesh topology (built once per plan).
//
// The fast forward kernel (dm_fast.cuh) walks the mesh as generalised triangle strips so that every per-vertex phase
// e^{-ik.v} is computed once per (frequency, strip visit) and shared by the up to three consecutive triangles that
// contain the vertex (north_star: "each vertex's phase ... reused across its incident triangles").  A strip is a vertex
// sequence s_0 s_1 s_2 ...; triangle i is (s_{i-2}, s_{i-1}, s_i).  One RECORD per sequence position:
//     vid_new[i]  the vertex entering at step i
//     vid_prev[i] the vertex that entered at step i-1        (edge e_i = v_new - v_prev)
//     vid_ret[i]  the vertex that entered at step i-2 and retires at step i (its phase is applied now)
//     fid[i]      the face (s_{i-2}, s_{i-1}, s_i), or -1 when the step closes no triangle (strip start / flush)
// Records are cut into n_chunks independent chunks (each starts with an empty window and ends with two flush
// records), every chunk padded to a multiple of DM_STRIP_UNROLL records.
#pragma once
#include <algorithm>
#include <cstdint>
#include <vector>

#define DM_STRIP_UNROLL 6

struct DmStripRecords {
    std::vector<int32_t> vid_new, vid_prev, vid_ret, fid;
    std::vector<int32_t> chunk_off;  // [n_chunks+1], record offsets
    int64_t n_strips = 0;
};

namespace dm_strips_detail {

struct Adj {
    // for face f and its edge j (opposite vertex j, i.e. edge (v_{j+1}, v_{j+2})): list of other faces on that edge
    std::vector<int32_t> off;   // [3*n_f+1]
    std::vector<int32_t> nbr;
};

inline Adj build_adjacency(const int32_t* faces, int32_t n_f, int32_t n_v)
{
    struct E { int64_t key; int32_t slot; };
    std::vector<E> es((size_t)n_f * 3);
    for (int32_t f = 0; f < n_f; ++f)
        for (int j = 0; j < 3; ++j) {
            int64_t a = faces[3 * f + (j + 1) % 3], b = faces[3 * f + (j + 2) % 3];
            if (a > b) std::swap(a, b);
            es[(size_t)3 * f + j] = {a * (int64_t)n_v + b, 3 * f + j};
        }
    std::sort(es.begin(), es.end(), [](const E& x, const E& y) { return x.key < y.key || (x.key == y.key && x.slot < y.slot); });
    Adj adj;
    adj.off.assign((size_t)n_f * 3 + 1, 0);
    size_t i = 0;
    while (i < es.size()) {
        size_t j = i;
        while (j < es.size() && es[j].key == es[i].key) ++j;
        for (size_t a = i; a < j; ++a) adj.off[(size_t)es[a].slot + 1] = (int32_t)(j - i - 1);
        i = j;
    }
    for (size_t s = 0; s < (size_t)n_f * 3; ++s) adj.off[s + 1] += adj.off[s];
    adj.nbr.resize((size_t)adj.off.back());
    std::vector<int32_t> fill(adj.off.begin(), adj.off.end() - 1);
    i = 0;
    while (i < es.size()) {
        size_t j = i;
        while (j < es.size() && es[j].key == es[i].key) ++j;
        for (size_t a = i; a < j; ++a)
            for (size_t b = i; b < j; ++b)
                if (a != b) adj.nbr[(size_t)fill[es[a].slot]++] = es[b].slot / 3;
        i = j;
    }
    return adj;
}

// the unvisited face across edge {a,b} of face f (other than f), or -1
inline int32_t across(const Adj& adj, const int32_t* faces, int32_t f, int32_t a, int32_t b,
                      const std::vector<int32_t>& state, int32_t stamp)
{
    for (int j = 0; j < 3; ++j) {
        const int32_t x = faces[3 * f + (j + 1) % 3], y = faces[3 * f + (j + 2) % 3];
        if ((x == a && y == b) || (x == b && y == a)) {
            for (int32_t q = adj.off[(size_t)3 * f + j]; q < adj.off[(size_t)3 * f + j + 1]; ++q) {
                const int32_t g = adj.nbr[q];
                if (state[g] == 0 || (state[g] < 0 && state[g] != -stamp)) return g;  // unvisited and not in this trial
            }
            return -1;
        }
    }
    return -1;
}

inline int32_t third_vertex(const int32_t* faces, int32_t g, int32_t a, int32_t b)
{
    for (int j = 0; j < 3; ++j) {
        const int32_t v = faces[3 * g + j];
        if (v != a && v != b) return v;
    }
    return -1;  // degenerate face (repeated vertex)
}

}  // namespace dm_strips_detail

// state[f]: 0 = unvisited, 1 = visited, negative = trial stamp
inline DmStripRecords dm_build_strips(const int32_t* faces, int32_t n_f, int32_t n_v, int n_chunks)
{
    using namespace dm_strips_detail;
    const Adj adj = build_adjacency(faces, n_f, n_v);
    std::vector<int32_t> state((size_t)n_f, 0);
    int32_t stamp = 1;
    struct Strip { std::vector<int32_t> verts, fids; };  // fids[i] = face closing at vertex i+2
    std::vector<Strip> strips;

    // walk from face f whose current last edge is (a,b); appends to verts/fids; marks faces with `mark`
    auto extend = [&](int32_t f, int32_t a, int32_t b, std::vector<int32_t>& verts, std::vector<int32_t>& fids, int32_t mark,
                      int32_t trial) {
        while (true) {
            const int32_t g = across(adj, faces, f, a, b, state, trial);
            if (g < 0) break;
            const int32_t c = third_vertex(faces, g, a, b);
            if (c < 0) break;
            state[g] = mark;
            verts.push_back(c);
            fids.push_back(g);
            f = g;
            a = b;
            b = c;
        }
    };

    for (int32_t seed = 0; seed < n_f; ++seed) {
        if (state[seed] == 1) continue;
        const int32_t v[3] = {faces[3 * seed], faces[3 * seed + 1], faces[3 * seed + 2]};
        if (v[0] == v[1] || v[1] == v[2] || v[0] == v[2]) {  // degenerate face: its own 3-vertex strip
            state[seed] = 1;
            strips.push_back({{v[0], v[1], v[2]}, {seed}});
            continue;
        }
        // try the three rotations of the seed (forward + backward extension) and keep the longest
        int best_rot = 0;
        size_t best_len = 0;
        for (int rot = 0; rot < 3; ++rot) {
            ++stamp;
            std::vector<int32_t> tv, tf;
            state[seed] = -stamp;
            extend(seed, v[(rot + 1) % 3], v[(rot + 2) % 3], tv, tf, -stamp, stamp);
            extend(seed, v[(rot + 1) % 3], v[rot], tv, tf, -stamp, stamp);
            if (rot == 0 || tf.size() > best_len) {
                best_len = tf.size();
                best_rot = rot;
            }
            state[seed] = 0;  // trial marks are negative stamps: they read as unvisited for later trials (see across())
        }
        // commit the best rotation: sequence (v[r], v[r+1], v[r+2], forward...) with a backward extension prepended
        ++stamp;
        const int r = best_rot;
        Strip s;
        state[seed] = 1;
        std::vector<int32_t> fv, ff, bv, bf;
        extend(seed, v[(r + 1) % 3], v[(r + 2) % 3], fv, ff, 1, stamp);
        // backward: strip read in reverse is (v[r+2], v[r+1], v[r], back...): last edge (v[r+1], v[r])
        extend(seed, v[(r + 1) % 3], v[r], bv, bf, 1, stamp);
        for (size_t i = bv.size(); i-- > 0;) s.verts.push_back(bv[i]);
        s.verts.push_back(v[r]);
        s.verts.push_back(v[(r + 1) % 3]);
        s.verts.push_back(v[(r + 2) % 3]);
        for (int32_t c : fv) s.verts.push_back(c);
        // faces in forward order: backward faces reversed (face closing at vertex i+2 of the reversed prefix), seed, forward
        for (size_t i = bf.size(); i-- > 0;) s.fids.push_back(bf[i]);
        s.fids.push_back(seed);
        for (int32_t g : ff) s.fids.push_back(g);
        strips.push_back(std::move(s));
    }

    // ---- chunks --------------------------------------------------------------------------------------------------
    DmStripRecords out;
    out.n_strips = (int64_t)strips.size();
    int64_t total = 0;
    for (const Strip& s : strips) total += (int64_t)s.verts.size();
    if (n_chunks < 1) n_chunks = 1;
    if ((int64_t)n_chunks > (int64_t)strips.size()) n_chunks = (int)std::max<size_t>(1, strips.size());
    out.chunk_off.push_back(0);
    size_t si = 0;
    int64_t done = 0;
    for (int c = 0; c < n_chunks; ++c) {
        const int64_t target = (total * (c + 1)) / n_chunks;
        int32_t last = -1;
        auto push = [&](int32_t vnew, int32_t vprev, int32_t vret, int32_t f) {
            out.vid_new.push_back(vnew);
            out.vid_prev.push_back(vprev);
            out.vid_ret.push_back(vret);
            out.fid.push_back(f);
        };
        int32_t p1 = -1, p2 = -1;  // vertices entered 1 and 2 steps ago (window), -1 = empty slot
        while (si < strips.size() && (done < target || c == n_chunks - 1)) {
            const Strip& s = strips[si++];
            for (size_t i = 0; i < s.verts.size(); ++i) {
                const int32_t vn = s.verts[i];
                push(vn, p1, p2, i >= 2 ? s.fids[i - 2] : -1);
                p2 = p1;
                p1 = vn;
                last = vn;
            }
            done += (int64_t)s.verts.size();
        }
        // two flush records retire the last two vertices; then pad to the unroll factor
        for (int k = 0; k < 2 || (out.fid.size() - (size_t)out.chunk_off.back()) % DM_STRIP_UNROLL != 0; ++k) {
            push(last, p1, p2, -1);
            p2 = p1;
            p1 = -1;  // nothing new enters: the slot stays empty so nothing is retired twice
        }
        out.chunk_off.push_back((int32_t)out.fid.size());
    }
    return out;
}
