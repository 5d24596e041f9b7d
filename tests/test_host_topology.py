"""Host logic of the CUDA library that needs no GPU: the triangle-strip walk of the forward kernel (dm_strips.h) and the
32-triangle patches of the backward kernel (dm_patches.h), compiled with g++ through tests/host/dump_topology.cpp and
checked for the invariants the kernels rely on."""
import os
import subprocess

import numpy as np
import pytest

from workloads import build_workload
from workloads.meshes import box_mesh

HERE = os.path.dirname(os.path.abspath(__file__))


@pytest.fixture(scope="module")
def dumper(tmp_path_factory):
    exe = tmp_path_factory.mktemp("host") / "dump_topology"
    subprocess.run(["g++", "-O2", "-std=c++17", "-o", str(exe), os.path.join(HERE, "host", "dump_topology.cpp")], check=True)
    return str(exe)


def _run(dumper, faces, n_v, tmp_path, n_chunks=4):
    src, dst = tmp_path / "faces.bin", tmp_path / "topo.txt"
    with open(src, "wb") as f:
        np.array([len(faces), n_v], dtype=np.int32).tofile(f)
        np.ascontiguousarray(faces, dtype=np.int32).tofile(f)
    subprocess.run([dumper, str(src), str(dst), str(n_chunks)], check=True)
    lines = open(dst).read().split("\n")
    n_p = int(lines[0].split()[1])
    pat = np.array([[int(x) for x in ln.split()] for ln in lines[1:1 + 32 * n_p]], dtype=np.int64)
    head = lines[1 + 32 * n_p].split()
    n_rec, n_ch = int(head[3]), int(head[5])
    off = np.array([int(x) for x in lines[2 + 32 * n_p:2 + 32 * n_p + n_ch + 1]])
    rec = np.array([[int(x) for x in ln.split()] for ln in lines[3 + 32 * n_p + n_ch:3 + 32 * n_p + n_ch + n_rec]], dtype=np.int64)
    return n_p, pat, off, rec


def _meshes():
    w2 = build_workload(2)
    w3 = build_workload(3, subdiv_override=2)      # 8 components of 320 faces
    vb, fb = box_mesh((0, 0, 0), (0.2, 0.3, 0.1))
    shuffled = w2.faces[np.random.default_rng(5).permutation(len(w2.faces))]
    open_mesh = w2.faces[:777]                      # a mesh with boundary
    return [("cfg2", w2.faces, len(w2.vertices)), ("aggregate", w3.faces, len(w3.vertices)), ("box", fb, len(vb)),
            ("shuffled", shuffled, len(w2.vertices)), ("open", open_mesh, len(w2.vertices))]


@pytest.mark.parametrize("name,faces,n_v", _meshes(), ids=lambda x: x if isinstance(x, str) else None)
def test_patches_partition_the_faces_and_index_their_vertices(dumper, tmp_path, name, faces, n_v):
    n_p, pat, _, _ = _run(dumper, faces, n_v, tmp_path)
    face, vid, loc = pat[:, 0], pat[:, 1], pat[:, 2]
    live = face >= 0
    assert sorted(face[live].tolist()) == list(range(len(faces)))          # every face exactly once
    for p in range(n_p):
        sl = slice(32 * p, 32 * p + 32)
        assert face[sl][0] >= 0                                              # lane 0 always holds a triangle
        v = vid[sl]
        used = v[v >= 0]
        assert len(set(used.tolist())) == len(used) <= 32                   # distinct vertices, one slot per lane
        assert (v[len(used):] == -1).all()
        for l in range(32):
            f = face[sl][l]
            if f < 0:
                continue
            slots = [(loc[sl][l] >> s) & 255 for s in (0, 8, 16)]
            assert [int(v[s]) for s in slots] == faces[f].tolist()          # corner slots point at the face's vertices
    if name in ("cfg2", "aggregate"):                                       # compact patches on the benchmark meshes
        idle = int((~live).sum())
        assert idle <= 0.03 * len(faces) + 31, idle
        per_patch = [int((vid[32 * p:32 * p + 32] >= 0).sum()) for p in range(n_p)]
        assert np.mean(per_patch) <= 30.5


@pytest.mark.parametrize("name,faces,n_v", _meshes(), ids=lambda x: x if isinstance(x, str) else None)
def test_strip_records_close_every_face_once_with_a_consistent_window(dumper, tmp_path, name, faces, n_v):
    _, _, off, rec = _run(dumper, faces, n_v, tmp_path, n_chunks=3)
    vnew, vprev, vret, fid = rec.T
    closed = fid[fid >= 0]
    assert sorted(closed.tolist()) == list(range(len(faces)))               # every face closed exactly once
    assert off[0] == 0 and off[-1] == len(rec) and (np.diff(off) % 6 == 0).all()
    for i in np.nonzero(fid >= 0)[0]:
        assert sorted([vnew[i], vprev[i], vret[i]]) == sorted(faces[fid[i]].tolist())
    # the window inside a chunk: prev / ret are what entered one / two steps ago (-1 = empty slot); the chunk ends with
    # flush records (no face, the last vertex repeated) during which nothing new enters
    for c in range(len(off) - 1):
        lo, hi = int(off[c]), int(off[c + 1])
        first_flush = hi
        while first_flush - 1 > lo and fid[first_flush - 1] < 0 and vnew[first_flush - 1] == vnew[first_flush - 2]:
            first_flush -= 1
        assert hi - first_flush >= 2                                        # the last two vertices are retired
        p1 = p2 = -1
        for i in range(lo, hi):
            assert vprev[i] == p1 and vret[i] == p2, (c, i)
            p2, p1 = p1, (vnew[i] if i < first_flush else -1)


# ---- k-splits of the backward (dm_splits.h) -----------------------------------------------------------------------------
@pytest.fixture(scope="module")
def split_dumper(tmp_path_factory):
    exe = tmp_path_factory.mktemp("host") / "dump_splits"
    subprocess.run(["g++", "-O2", "-std=c++17", "-o", str(exe), os.path.join(HERE, "host", "dump_splits.cpp")], check=True)
    return str(exe)


def _splits(exe, nx, ny, nzh, n_faces, n_sm=148, band=0, slab=None):
    args = [exe, str(nx), str(ny), str(nzh), str(n_faces), str(n_sm), str(band)]
    if slab is not None:
        args += [str(slab[0]), str(slab[1])]
    out = subprocess.run(args, check=True, capture_output=True, text=True).stdout.split()
    return tuple(int(x) for x in out)   # n_split_max, n_split, rows_per_split


def test_backward_splits_never_outgrow_the_fast_kernels_row_index(split_dumper):
    """A split holds at most 32768 rows (the fast backward kernel's 15-bit row index), whatever the mesh and grid: a huge
    mesh (few splits wanted) on a wide grid used to get one split of nx*ny rows and fell back to the robust kernel."""
    cases = [(4096, 64, 33, 4_000_000), (4096, 4096, 2, 5_000_000), (512, 512, 257, 3_600_000), (4096, 4096, 2, 320),
             (128, 128, 65, 102_400), (256, 256, 129, 327_680), (32, 32, 17, 320), (2, 2, 2, 12)]
    for nx, ny, nzh, n_faces in cases:
        for band in (0, 1):
            n_max, n_split, rps = _splits(split_dumper, nx, ny, nzh, n_faces, band=band)
            n_rows = nx * ny
            assert 1 <= n_split <= n_max, (nx, ny, nzh, n_faces)
            assert rps <= 32768, (nx, ny, nzh, n_faces, rps)
            assert (n_split - 1) * rps < n_rows <= n_split * rps       # the splits tile the rows, none is empty
            assert n_max * 13 * n_faces <= max(64 * 13 * n_faces, (n_rows + 32767) // 32768 * 13 * n_faces, 64 << 20)
    # the case of the report: ~4 M faces, 262144 rows -> 8 splits of 32768 rows rather than 1 of 262144
    assert _splits(split_dumper, 4096, 64, 33, 4_000_000)[1:] == (8, 32768)
    # x-slabs keep the bound too
    assert _splits(split_dumper, 4096, 4096, 2, 4_000_000, slab=(0, 2048))[2] <= 32768


def test_backward_splits_of_the_bench_configs_are_unchanged(split_dumper):
    """The fix must not move the launch configuration bench.py times (cfg 4: 128^3, 102400 triangles; cfg 5: 256^3, 327680)."""
    assert _splits(split_dumper, 128, 128, 65, 102_400) == (64, 36, 456)
    assert _splits(split_dumper, 256, 256, 129, 327_680) == (64, 12, 5462)
