"""mesh_voxel.py — TEST INFRASTRUCTURE, NOT THE PRODUCT.  CPU oracle of the triangle-mesh voxeliser.

What it follows.  PAPER.md:191 (§3.1): "We re-voxelize the triangle mesh by casting axis-aligned rays through grid columns
and computing ray-triangle intersections, using an odd-even parity rule along each column.  To improve robustness near
degeneracies, we corroborate independent passes along different ray directions for solid labeling."  PAPER.md:51: "A
ray-tracing-based occupancy test efficiently classifies solid and fluid cells".  The paper gives no tie rules; the
reading (DESIGN.md §4 reading 22) is written out below, in exact integer arithmetic so that the labels are unique:

  * Mesh coordinates are lattice units (cell (x,y,z) has its centre at (x+1/2, y+1/2, z+1/2)).  Vertices are snapped to
    1/256 of a cell: v = rint(float32(coord) * 256) (round half to even), an integer; they must lie in [-2^18, 2^19).
  * Pass d (d = x, y, z): the ray runs along axis d through the cell centres of a grid column.  With (u, v) the other two
    axes in cyclic order ((y,z) for x, (z,x) for y, (x,y) for z), a triangle is hit by the ray at P = (pu, pv) iff P lies
    inside its projection on the (u,v) plane.  Projections of zero area are skipped.  The projection is taken
    counter-clockwise (two vertices swapped if its area is negative); P on an edge a->b counts as inside iff the edge
    direction (du, dv) has dv < 0, or dv = 0 and du > 0 (the "top-left" rule: a shared edge belongs to exactly one of
    the two triangles beside it, so a ray through an edge or a vertex is counted once).
  * The crossing lies at w* = interpolated d-coordinate of the plane at P (an exact rational).  It flips the parity of
    every cell of the column whose centre is at or beyond it: centre_w >= w*  (with the edge rule above this makes every
    axis half-open the same way in all three passes: a centre exactly on the low face of a box is inside, on the high
    face outside).
  * parity_d(cell) = number of crossings with w* <= centre_w, mod 2.  Label: SOLID iff at least `min_votes` of the three
    passes say odd (2 = majority, the "corroboration" of PAPER.md:191).

Deliberately slow and plain: a Python loop over triangles, numpy int64 over the columns of each triangle's bounding box,
floor divisions exactly as written above.  Pins: tests/test_oracle_mesh.py (closed-form boxes, integer translation,
additivity of adjacent boxes, agreement with an independent winding-number test, holes repaired by the vote, prisms =
the heightmap voxeliser).  Shares nothing with paper_2607_04516_b200/.
"""
from __future__ import annotations

import numpy as np

SUB = 256           # sub-units per cell
LO, HI = -(1 << 18), (1 << 19)


def snap(tri) -> np.ndarray:
    """float coordinates [n][3][3] (lattice units) -> integer sub-units, int64."""
    t = np.asarray(tri, dtype=np.float32).reshape(-1, 3, 3)
    v = np.rint(t * np.float32(SUB)).astype(np.int64)
    if v.size and (v.min() < LO or v.max() >= HI):
        raise ValueError("mesh vertex outside [-1024, 2048) cells")
    return v


def _pass_parity(v: np.ndarray, shape, d: int) -> np.ndarray:
    """parity_d for all cells; shape = (nx, ny, nz); returns uint8 [nz][ny][nx]."""
    n = (shape[0], shape[1], shape[2])
    au, av, aw = (d + 1) % 3, (d + 2) % 3, d
    nu, nv, nw = n[au], n[av], n[aw]
    toggles = np.zeros((nu, nv, nw + 1), dtype=np.int64)     # [u][v][k]; slot nw collects crossings beyond the column
    for t in v:
        a, b, c = t[0], t[1], t[2]
        area = (b[au] - a[au]) * (c[av] - a[av]) - (b[av] - a[av]) * (c[au] - a[au])
        if area == 0:
            continue
        if area < 0:
            b, c = c, b
            area = -area
        # columns whose centre can lie inside: centre_u = (2 iu + 1) * 128
        umin, umax = min(a[au], b[au], c[au]), max(a[au], b[au], c[au])
        vmin, vmax = min(a[av], b[av], c[av]), max(a[av], b[av], c[av])
        iu0, iu1 = max(0, (umin - 128) // 256), min(nu - 1, (umax - 128) // 256 + 1)
        iv0, iv1 = max(0, (vmin - 128) // 256), min(nv - 1, (vmax - 128) // 256 + 1)
        if iu0 > iu1 or iv0 > iv1:
            continue
        pu = ((2 * np.arange(iu0, iu1 + 1, dtype=np.int64) + 1) * 128)[:, None]
        pv = ((2 * np.arange(iv0, iv1 + 1, dtype=np.int64) + 1) * 128)[None, :]

        def edge(p, q):
            du, dv = q[au] - p[au], q[av] - p[av]
            e = du * (pv - p[av]) - dv * (pu - p[au])
            incl = (dv < 0) or (dv == 0 and du > 0)
            return e, (e > 0) | ((e == 0) & incl)

        wa, ina = edge(b, c)       # weight of vertex a = edge function of the opposite edge
        wb, inb = edge(c, a)
        wc, inc = edge(a, b)
        inside = ina & inb & inc
        if not inside.any():
            continue
        # w* = (wa a_w + wb b_w + wc c_w) / area ;  cell k is at or beyond the crossing iff (2k+1) 128 area >= numerator
        num = wa * a[aw] + wb * b[aw] + wc * c[aw]
        q = -np.floor_divide(-num, 128 * area)               # ceil(w* / 128)
        k = np.floor_divide(q, 2)                            # smallest k with 2k+1 >= w*/128
        k = np.clip(k, 0, nw)
        iu, iv = np.nonzero(inside)
        np.add.at(toggles, (iu + iu0, iv + iv0, k[iu, iv]), 1)
    par = (np.cumsum(toggles[:, :, :nw], axis=2) & 1).astype(np.uint8)   # [u][v][w]
    # back to [z][y][x]
    axes = [0, 0, 0]
    axes[au], axes[av], axes[aw] = 0, 1, 2                   # par's axis holding x, y, z respectively
    return np.ascontiguousarray(par.transpose(axes[2], axes[1], axes[0]))


def pass_parities(tri, nx, ny, nz):
    """The three passes separately: (parity_x, parity_y, parity_z), each uint8 [nz][ny][nx]."""
    v = snap(tri)
    return tuple(_pass_parity(v, (nx, ny, nz), d) for d in range(3))


def voxelise(tri, nx, ny, nz, min_votes=2) -> np.ndarray:
    """SOLID mask uint8 [nz][ny][nx]: at least min_votes of the three ray directions say 'inside'."""
    px, py, pz = pass_parities(tri, nx, ny, nz)
    return ((px.astype(np.int32) + py + pz) >= min_votes).astype(np.uint8)
