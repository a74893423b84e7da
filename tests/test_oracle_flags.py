"""Pins for the integer work of the oracle: voxelisation and link classification.

The brute force here is a different formulation from the oracle's per-axis resolve(): it builds the
domain with one explicit ghost layer per face (periodic -> wrapped copy, wall -> solid, free-slip -> copy of
the boundary layer, i.e. the mirror image) and says "link i of a fluid cell is a wall link iff the ghost-
extended cell at x - c_i is solid".
"""
import itertools

import numpy as np
import pytest

import oracle
from oracle import Oracle

P, WALL, FS, EQF, EQO = 0, 1, 2, 3, 4
FLUID, SOLID, C_EQF, C_EQO = 0, 1, 2, 3


def brute_flags(hm, nz, faces):
    ny, nx = hm.shape
    cls = np.zeros((nz, ny, nx), dtype=np.uint8)
    for z, y, x in itertools.product(range(nz), range(ny), range(nx)):
        if z < min(max(int(hm[y, x]), 0), nz):
            cls[z, y, x] = SOLID
            continue
        on = [x == 0, x == nx - 1, y == 0, y == ny - 1, z == 0, z == nz - 1]
        types = {faces[k] for k in range(6) if on[k]}
        if EQF in types:
            cls[z, y, x] = C_EQF
        elif EQO in types:
            cls[z, y, x] = C_EQO
    return cls


def _ghost_extend(solid, faces):
    """solid[z][y][x] -> array with one ghost layer on every side."""
    out = solid
    for axis, (lo, hi) in zip((2, 1, 0), ((faces[0], faces[1]), (faces[2], faces[3]), (faces[4], faces[5]))):
        first = np.take(out, [0], axis=axis)
        last = np.take(out, [-1], axis=axis)

        def ghost(ft, wrapped, edge):
            if ft == P:
                return wrapped
            if ft == WALL:
                return np.ones_like(edge)
            if ft == FS:
                return edge
            return np.zeros_like(edge)  # EQ faces: never reached from a FLUID cell

        out = np.concatenate([ghost(lo, last, first), out, ghost(hi, first, last)], axis=axis)
    return out


def brute_links(cls, faces):
    c, _, _ = oracle.lattice()
    nz, ny, nx = cls.shape
    ext = _ghost_extend(cls == SOLID, faces)
    links = np.zeros(cls.shape, dtype=np.uint32)
    for z, y, x in itertools.product(range(nz), range(ny), range(nx)):
        if cls[z, y, x] != FLUID:
            continue
        bits = 0
        for i in range(1, 19):
            if ext[z - c[i, 2] + 1, y - c[i, 1] + 1, x - c[i, 0] + 1]:
                bits |= 1 << i
        links[z, y, x] = bits
    return links


FACE_SETS = [
    (P, P, P, P, P, P),
    (EQF, EQO, P, P, WALL, FS),          # config 1
    (EQF, EQO, FS, FS, WALL, FS),        # config 3
    (EQF, EQO, EQF, EQF, WALL, FS),      # config 4
    (P, P, P, P, WALL, FS),              # config 5 precursor
    (WALL, WALL, WALL, WALL, WALL, WALL),
    (FS, FS, FS, FS, FS, FS),
    (FS, WALL, P, P, FS, WALL),
    (EQO, EQF, WALL, FS, P, P),
]


@pytest.mark.parametrize("faces", FACE_SETS)
def test_flags_and_links_match_brute_force_on_small_boxes(faces):
    rng = np.random.default_rng(hash(faces) % (2 ** 32))
    for nx, ny, nz in [(6, 5, 4), (8, 8, 8), (3, 4, 7)]:
        hm = rng.integers(-1, nz + 2, size=(ny, nx)).astype(np.int32)
        hm[rng.random((ny, nx)) < 0.5] = 0
        o = Oracle(nx, ny, nz, 1e-3, 0.1, 0.0, (0, 0, 0), faces)
        o.set_flags(hm)
        cls = o.get_flags()
        np.testing.assert_array_equal(cls, brute_flags(hm, nz, faces))
        assert int((cls == SOLID).sum()) == int(np.clip(hm, 0, nz).sum())
        np.testing.assert_array_equal(o.get_links(), brute_links(cls, faces))


def test_links_in_a_periodic_box_are_symmetric_under_direction_reversal():
    """#(fluid cell, direction i) wall links == #(fluid cell, opposite i) wall links in a fully periodic box:
    every fluid->solid lattice edge is seen once from each side of the solid."""
    _, _, opp = oracle.lattice()
    rng = np.random.default_rng(0)
    hm = (rng.random((12, 14)) < 0.3) * rng.integers(1, 9, size=(12, 14))
    o = Oracle(14, 12, 9, 1e-3, 0.0, 0.0, (0, 0, 0), (P,) * 6)
    o.set_flags(hm.astype(np.int32))
    links = o.get_links()
    counts = [int(((links >> i) & 1).sum()) for i in range(19)]
    assert counts[0] == 0
    # heightmap solids are columns: a link along +c and one along -c exist in equal number only for
    # directions with c_z = 0 or when summed with their z-mirror; reversal symmetry holds for every i in x,y
    for i in range(1, 19):
        c = oracle.lattice()[0]
        if c[i, 2] == 0:
            assert counts[i] == counts[opp[i]]


def test_config1_flags():
    from paper_2607_04516_b200 import workloads as W
    wl = W.config1()
    o = Oracle(wl.nx, wl.ny, wl.nz, wl.nu0, wl.Cs, wl.f_cor, wl.F, wl.faces)
    o.set_flags(wl.height)
    cls = o.get_flags()
    assert (cls == SOLID).sum() == 8 * 8 * 16
    assert (cls[:, :, 0] == C_EQF).all() and (cls[:, :, -1] == C_EQO).all()
    assert (cls[:, :, 1:-1] >= C_EQF).sum() == 0
    links = o.get_links()
    # ground: every fluid cell of level 0 has exactly the 5 downward-pulling links (c_z = +1 arrive from below)
    c = oracle.lattice()[0]
    up = sum(1 << i for i in range(19) if c[i, 2] == 1)
    free = cls[0] == FLUID
    away = np.ones_like(free)
    away[11:21, 15:25] = False
    assert np.all(links[0][free & away] == up)
    # top is free-slip: no wall links on the top level away from the building
    assert np.all(links[-1][cls[-1] == FLUID] == 0)
