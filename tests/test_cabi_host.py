"""CPU-only checks of the C-ABI library (no compute calls, no GPU): it loads, exports every symbol that
include/qxd.h declares, rejects bad geometry, and its on-the-fly site order (PAPER.md:97,105,
137-139) is a bijection whose neighbour function agrees with an independent numpy neighbour table."""
import ctypes as C
import os
import re

import numpy as np
import pytest

import lattice_np as LN

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2502_02490_b200 import build, binding
    build.build()
    return binding.load_library()


def declared_functions():
    src = open(os.path.join(ROOT, "include", "qxd.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(qxd_[a-z0-9_A-Z]+)\s*\(", src)))


def test_every_declared_symbol_is_exported_and_bound(lib):
    from paper_2502_02490_b200 import binding
    names = declared_functions()
    assert len(names) >= 25
    for n in names:
        assert hasattr(lib, n), f"libqxd.so does not export {n}"
        assert n in binding.SYMBOLS, f"binding.py does not declare {n}"
    assert set(binding.SYMBOLS) == set(names)
    assert lib.qxd_version().decode().startswith("qxd-b200")


def test_pairing_needs_cstar(lib):
    h = C.c_void_p()
    assert lib.qxd_geometry_create(4, 4, 4, 4, 4, C.byref(h)) == 0
    assert lib.qxd_set_cstar_pairing(h, 1) == -1
    lib.qxd_geometry_destroy(h)


def test_geometry_argument_checks(lib):
    h = C.c_void_p()
    for bad in ((3, 4, 4, 4, 0), (4, 4, 4, 0, 0), (4, 2, 4, 5, 1), (4, 4, 4, 4, 8), (4, 4, 4, 4, -1)):
        assert lib.qxd_geometry_create(*bad, C.byref(h)) == -1 and not h.value
    assert lib.qxd_geometry_create(4, 2, 2, 6, 3 | 4, C.byref(h)) == 0
    assert lib.qxd_volume(h) == 4 * 4 * 2 * 6
    assert lib.qxd_set_tile(h, 2, 2, 2, 1) == -1           # b3 must be >= 2
    assert lib.qxd_set_tile(h, 3, 2, 2, 2) == -1           # not a power of two
    assert lib.qxd_set_tile(h, 2, 2, 2, 2) == 0
    assert lib.qxd_workspace_bytes(h, 1, 1) > 0
    assert lib.qxd_workspace_bytes(h, 7, 1) > lib.qxd_workspace_bytes(h, 1, 1)
    # state errors need no GPU: nothing is bound yet
    assert lib.qxd_set_quark(h, 0.12, 0.0) == -2
    assert lib.qxd_clover_build(h, 1.0, 0.0) == -2
    assert lib.qxd_geometry_destroy(h) == 0


@pytest.mark.parametrize("dims,cstar,tile,block,pairing", [
    ((4, 4, 4, 4), 0, None, None, 0),
    ((8, 4, 4, 8), 3, None, None, 0),
    ((8, 2, 6, 4), 2, (2, 2, 2, 4), (4, 4, 2, 4), 0),
    ((16, 4, 4, 4), 1, (4, 4, 4, 4), (16, 4, 4, 4), 0),
    ((6, 2, 2, 2), 3, None, None, 0),
    # C*-paired layout: (physical site, mirror bit); same extended-lattice neighbour relation
    ((8, 4, 4, 8), 3, None, None, 1),
    ((8, 2, 6, 4), 2, (2, 2, 2, 4), (4, 2, 2, 4), 1),
    ((16, 4, 4, 4), 1, None, None, 1),
    ((6, 2, 2, 2), 3, None, None, 1),
])
def test_site_order_bijection_and_neighbours(lib, dims, cstar, tile, block, pairing):
    h = C.c_void_p()
    assert lib.qxd_geometry_create(*dims, cstar | 4, C.byref(h)) == 0
    if cstar:
        assert lib.qxd_set_cstar_pairing(h, pairing) == 0     # the paired layout is the default for C* geometries
    if tile:
        assert lib.qxd_set_tile(h, *tile) == 0
    if block:
        assert lib.qxd_set_block(h, *block) == 0
    lat = LN.Lattice(*dims, cstar=cstar)
    V = lat.V
    assert lib.qxd_volume(h) == V
    I4 = C.c_int * 4
    cb, par, nb = C.c_int(), C.c_int(), C.c_int()
    index = np.empty((V, 2), dtype=np.int64)
    for s in range(V):
        x = I4(*[int(v) for v in lat.coords[s]])
        assert lib.qxd_site_index(h, x, C.byref(cb), C.byref(par)) == 0
        index[s] = (cb.value, par.value)
        y = I4()
        assert lib.qxd_site_coords(h, cb.value, par.value, y) == 0
        assert list(y) == list(x)
    assert np.array_equal(index[:, 1], lat.parity)                       # parity from extended coordinates
    for p in (0, 1):                                                     # each parity fills [0, V/2) exactly once
        assert sorted(index[index[:, 1] == p, 0]) == list(range(V // 2))
    for s in range(V):
        for mu in range(4):
            for d, step in enumerate((+1, -1)):
                assert lib.qxd_site_neighbour(h, int(index[s, 0]), int(index[s, 1]), mu, step, C.byref(nb)) == 0
                t = lat.nbr[mu, d, s]
                assert index[t, 1] == 1 - index[s, 1]
                assert nb.value == index[t, 0], (s, mu, step)
    if pairing:   # a site and its mirror image x + L1 e1 are consecutive indices of the same parity
        L1 = dims[1]
        for s in range(V):
            x = lat.coords[s]
            if x[1] < L1:
                y = I4(int(x[0]), int(x[1]) + L1, int(x[2]), int(x[3]))
                assert lib.qxd_site_index(h, y, C.byref(cb), C.byref(par)) == 0
                assert (cb.value, par.value) == (int(index[s, 0]) + 1, int(index[s, 1])) and index[s, 0] % 2 == 0
    assert lib.qxd_site_neighbour(h, 0, 0, 4, 1, C.byref(nb)) == -1
    assert lib.qxd_site_coords(h, V // 2, 0, I4()) == -1
    lib.qxd_geometry_destroy(h)


@pytest.mark.parametrize("dims,cstar,pairing,ok", [
    ((8, 8, 8, 8), 0, 0, True),
    ((8, 8, 8, 8), 3, 0, True),       # extended layout, L1 / 4 even: the C* shift keeps the direction-1 colour
    ((8, 4, 8, 8), 3, 0, False),      # L1 / 4 odd: a hop across a C* boundary would land on the same colour -> rejected
    ((8, 4, 8, 8), 3, 1, True),       # paired layout: the shift is a flip of the mirror bit inside the block
    ((16, 8, 4, 8), 2, 1, True),      # a single block in a C* direction (paired: the wrap stays inside the block)
    ((12, 4, 4, 4), 0, 0, False),     # three blocks in time
    ((4, 4, 4, 4), 0, 0, False),      # one tile: an odd number of tiles
])
def test_sap_blocks_are_two_coloured(lib, dims, cstar, pairing, ok):
    """Reading R21 on the host (no GPU): blocks are the 128-index tiles of both parities; whenever a hop leaves a block it
    lands on a block of the other colour, for every site and direction including the shifted C* wraps; geometries without
    such a colouring are rejected."""
    h = C.c_void_p()
    assert lib.qxd_geometry_create(*dims, cstar | 4, C.byref(h)) == 0
    if cstar:
        assert lib.qxd_set_cstar_pairing(h, pairing) == 0
    V = lib.qxd_volume(h)
    blk, col, nb = C.c_int(), C.c_int(), C.c_int()
    rc = lib.qxd_sap_block_of(h, 0, 0, C.byref(blk), C.byref(col))
    if not ok:
        assert rc == -1 and b"two-colouring" in lib.qxd_last_error(h)
        lib.qxd_geometry_destroy(h)
        return
    assert rc == 0
    info = {}
    for p in (0, 1):
        for cb in range(V // 2):
            assert lib.qxd_sap_block_of(h, cb, p, C.byref(blk), C.byref(col)) == 0
            assert blk.value == cb >> 7
            info[(cb, p)] = (blk.value, col.value)
    colour_of_block = {}
    for (b, c) in info.values():
        assert colour_of_block.setdefault(b, c) == c                       # one colour per block, both parities
    counts = [list(colour_of_block.values()).count(k) for k in (0, 1)]
    assert counts[0] == counts[1] == V // 512                              # half of the blocks each
    for j in range(V // 512):                                              # the kernel's pairing of consecutive tiles
        assert colour_of_block[2 * j] != colour_of_block[2 * j + 1]
    crossings = 0
    for (cb, p), (b, c) in info.items():
        for mu in range(4):
            for step in (+1, -1):
                assert lib.qxd_site_neighbour(h, cb, p, mu, step, C.byref(nb)) == 0
                b2, c2 = info[(nb.value, 1 - p)]
                if b2 != b:
                    crossings += 1
                    assert c2 != c, (cb, p, mu, step)
    assert crossings > 0
    lib.qxd_geometry_destroy(h)


def test_solver_space_setters_check_their_arguments(lib):
    """qxd_set_gcr / qxd_set_deflation / qxd_set_deflation_chirality / qxd_set_deflation_refine: host-side argument checks (no GPU
    needed: the solver spaces are only carved at qxd_workspace_bind)."""
    h = C.c_void_p()
    assert lib.qxd_geometry_create(8, 8, 8, 8, 4, C.byref(h)) == 0
    assert lib.qxd_set_gcr(h, 16, 4, 5) == 0
    assert lib.qxd_set_gcr(h, 33, 4, 5) == -1
    assert lib.qxd_set_deflation(h, 24, 8, 12, 0) == 0
    assert lib.qxd_set_deflation(h, 7, 8, 12, 0) == -1                 # odd number of null vectors
    assert lib.qxd_set_deflation(h, 34, 8, 12, 0) == -1
    assert lib.qxd_set_deflation_chirality(h, 1) == -1                 # 24 vectors would be 48 coarse degrees of freedom per block
    assert b"16" in lib.qxd_last_error(h)
    assert lib.qxd_set_deflation(h, 16, 8, 12, 0) == 0
    assert lib.qxd_set_deflation_chirality(h, 1) == 0
    assert lib.qxd_set_deflation(h, 18, 8, 12, 0) == -1                # and the other way round
    assert lib.qxd_set_deflation_chirality(h, 2) == -1
    assert lib.qxd_set_deflation_refine(h, 2, 4) == 0
    assert lib.qxd_set_deflation_refine(h, -1, 4) == -1
    assert lib.qxd_set_deflation_refine(h, 1, 0) == -1 and lib.qxd_set_deflation_refine(h, 1, 17) == -1
    nb, ns, ready = C.c_int(), C.c_int(), C.c_int()
    assert lib.qxd_deflation_info(h, C.byref(nb), C.byref(ns), C.byref(ready)) == 0
    assert (nb.value, ns.value, ready.value) == (8 * 8 * 8 * 8 // 256, 32, 0)
    assert lib.qxd_geometry_destroy(h) == 0
