"""Pins for the oracle's triangle-mesh voxeliser (oracle/mesh_voxel.py; "casting axis-aligned rays through
grid columns and computing ray-triangle intersections, using an odd-even parity rule along each column ... corroborate
independent passes along different ray directions"; PAPER.md:51 Boolean merge of base, terrain and building layers).

None of these re-types the ray casting: closed-form cell sets of boxes, an independent point-in-polyhedron test (solid
angle / winding number in float64), integer translation, additivity of boxes sharing a face (internal faces cancel),
degenerate placements (faces, edges and vertices exactly on cell centres), holes repaired by the vote, extruded
footprints = the heightmap voxeliser."""
import numpy as np
import pytest


@pytest.fixture(scope="module")
def MV(oracle_mod):
    return oracle_mod.mesh_voxel


@pytest.fixture(scope="module")
def W():
    from paper_2607_04516_b200 import workloads
    return workloads


def centres_inside_box(lo, hi, nx, ny, nz, closed_lo=False):
    z, y, x = np.meshgrid(np.arange(nz) + 0.5, np.arange(ny) + 0.5, np.arange(nx) + 0.5, indexing="ij")
    c = (x, y, z)
    m = np.ones((nz, ny, nx), bool)
    for a in range(3):
        m &= (c[a] >= lo[a]) if closed_lo else (c[a] > lo[a])
        m &= c[a] < hi[a]
    return m.astype(np.uint8)


def solid_angle_inside(tri, pts):
    """Winding number of a closed mesh about each point (van Oosterom-Strackee), float64; True where |w| > 1/2."""
    t = np.asarray(tri, dtype=np.float64)
    w = np.zeros(len(pts))
    for a, b, c in t:
        ra, rb, rc = a - pts, b - pts, c - pts
        la, lb, lc = [np.linalg.norm(r, axis=1) for r in (ra, rb, rc)]
        num = np.einsum("ij,ij->i", ra, np.cross(rb, rc))
        den = la * lb * lc + np.einsum("ij,ij->i", ra, rb) * lc + np.einsum("ij,ij->i", rb, rc) * la + np.einsum("ij,ij->i", rc, ra) * lb
        w += 2.0 * np.arctan2(num, den)
    return np.abs(w / (4 * np.pi)) > 0.5


def test_box_with_generic_coordinates_is_the_set_of_cell_centres_inside(MV, W):
    nx, ny, nz = 11, 9, 7
    rng = np.random.default_rng(1)
    for _ in range(20):
        lo = rng.uniform(-2, 5, 3)
        hi = lo + rng.uniform(0.3, 7, 3)
        lo, hi = np.round(lo * 256 + 0.37) / 256, np.round(hi * 256 + 0.37) / 256   # on the 1/256 grid, never on a centre plane
        want = centres_inside_box(lo, hi, nx, ny, nz)
        px, py, pz = MV.pass_parities(W.box_mesh(lo, hi), nx, ny, nz)
        for p in (px, py, pz):
            np.testing.assert_array_equal(p, want)
        np.testing.assert_array_equal(MV.voxelise(W.box_mesh(lo, hi), nx, ny, nz), want)


def test_faces_edges_and_vertices_exactly_on_cell_centres(MV, W):
    """Box corners at half-integers: every ray of the boundary columns runs through edges / vertices of the triangulated
    faces.  The tie rules make each pass count such a ray once, all three passes agree, and the result is a box of cells
    whose volume is exactly the box volume (half-open in every axis), shifted consistently."""
    nx, ny, nz = 10, 9, 8
    lo, hi = (1.5, 2.5, 1.5), (6.5, 5.5, 4.5)
    px, py, pz = MV.pass_parities(W.box_mesh(lo, hi), nx, ny, nz)
    np.testing.assert_array_equal(px, py)
    np.testing.assert_array_equal(py, pz)
    assert int(px.sum()) == 5 * 3 * 3
    idx = np.argwhere(px)
    assert tuple(idx.max(0) - idx.min(0) + 1) == (3, 3, 5)
    # integer translation of the mesh translates the labels
    q = MV.voxelise(W.box_mesh((2.5, 4.5, 2.5), (7.5, 7.5, 5.5)), nx, ny, nz)
    np.testing.assert_array_equal(q[1:, 2:, 1:], px[:-1, :-2, :-1])
    assert q.sum() == px.sum()


def test_adjacent_boxes_add_up_and_their_shared_face_cancels(MV, W):
    nx, ny, nz = 12, 8, 8
    for cut in (4.0, 4.5, 4.3):          # the shared face between cells, through cell centres, generic
        a = W.box_mesh((1.25, 1.5, 0.75), (cut, 6.25, 5.5))
        b = W.box_mesh((cut, 1.5, 0.75), (9.75, 6.25, 5.5))
        whole = W.box_mesh((1.25, 1.5, 0.75), (9.75, 6.25, 5.5))
        va, vb = MV.voxelise(a, nx, ny, nz), MV.voxelise(b, nx, ny, nz)
        vw = MV.voxelise(whole, nx, ny, nz)
        assert not (va & vb).any()                                             # no cell claimed twice
        np.testing.assert_array_equal(va | vb, vw)
        np.testing.assert_array_equal(MV.voxelise(np.concatenate([a, b]), nx, ny, nz), vw)   # one mesh with an internal wall


def test_sphere_agrees_with_the_winding_number_and_with_its_volume(MV, W):
    nx, ny, nz = 24, 22, 20
    c, r = (11.3, 10.6, 9.8), 7.7
    tri = W.icosphere_mesh(c, r, 2)
    px, py, pz = MV.pass_parities(tri, nx, ny, nz)
    np.testing.assert_array_equal(px, py)
    np.testing.assert_array_equal(py, pz)
    z, y, x = np.meshgrid(np.arange(nz) + 0.5, np.arange(ny) + 0.5, np.arange(nx) + 0.5, indexing="ij")
    pts = np.stack([x.ravel(), y.ravel(), z.ravel()], axis=1)
    snapped = MV.snap(tri).astype(np.float64) / 256.0
    want = solid_angle_inside(snapped, pts).reshape(nz, ny, nx)
    np.testing.assert_array_equal(px.astype(bool), want)
    # polyhedron volume (divergence theorem) vs cell count: within the surface-cell uncertainty
    vol = abs(sum(np.dot(a, np.cross(b, cc)) for a, b, cc in snapped)) / 6.0
    assert abs(px.sum() - vol) < 0.03 * vol
    assert vol == pytest.approx(4 / 3 * np.pi * r ** 3, rel=0.05)


def test_a_hole_breaks_one_pass_and_the_vote_repairs_it(MV, W):
    nx, ny, nz = 10, 10, 10
    lo, hi = (2.25, 2.25, 1.25), (7.75, 7.75, 6.75)
    tri = W.box_mesh(lo, hi)
    want = centres_inside_box(lo, hi, nx, ny, nz)
    top = [i for i, t in enumerate(tri) if np.all(t[:, 2] == np.float32(hi[2]))]
    assert len(top) == 2
    holed = np.delete(tri, top[0], axis=0)                    # half of the roof missing
    px, py, pz = MV.pass_parities(holed, nx, ny, nz)
    np.testing.assert_array_equal(px, want)                   # horizontal rays never meet the roof
    np.testing.assert_array_equal(py, want)
    assert (pz != want).any()                                 # vertical rays under the hole leak to the top of the box
    leak = np.argwhere(pz != want)
    assert (leak[:, 0] > 6).all()                             # ... above the roof only
    np.testing.assert_array_equal(MV.voxelise(holed, nx, ny, nz, 2), want)
    assert MV.voxelise(holed, nx, ny, nz, 3).sum() == want.sum()      # unanimity loses nothing here: the leak is outside
    assert MV.voxelise(holed, nx, ny, nz, 1).sum() > want.sum()       # any-vote keeps the leak


def test_extruded_footprints_equal_the_heightmap_voxeliser_and_merge_with_terrain(MV, W, oracle_mod):
    nx, ny, nz = 40, 30, 16
    hm = W.urban_heightmap(nx, ny, seed=7)
    hm = np.minimum(hm, nz - 3).astype(np.int32)
    tri = W.urban_mesh(hm)
    mask = MV.voxelise(tri, nx, ny, nz)
    z = np.arange(nz)[:, None, None]
    np.testing.assert_array_equal(mask, (z < hm[None]).astype(np.uint8))
    # Boolean merge: base layer of 1 cell + terrain ramp as a heightmap, buildings as a mesh standing on it
    terrain = (1 + (np.arange(nx)[None, :] // 10) + 0 * np.arange(ny)[:, None]).astype(np.int32)
    o1 = oracle_mod.Oracle(nx, ny, nz, 1e-2, 0.1, 0.0, (0, 0, 0), (3, 4, 0, 0, 1, 2))
    o1.set_flags_mask(terrain, mask)
    o2 = oracle_mod.Oracle(nx, ny, nz, 1e-2, 0.1, 0.0, (0, 0, 0), (3, 4, 0, 0, 1, 2))
    o2.set_flags(np.maximum(terrain, hm))
    np.testing.assert_array_equal(o1.get_flags(), o2.get_flags())
    np.testing.assert_array_equal(o1.get_links(), o2.get_links())
    # an overhang (a slab on two legs) cannot be a heightmap: mask only
    bridge = np.concatenate([W.box_mesh((5.2, 5.2, -1), (7.8, 9.8, 8.6)), W.box_mesh((15.2, 5.2, -1), (17.8, 9.8, 8.6)),
                             W.box_mesh((5.2, 5.2, 6.4), (17.8, 9.8, 8.6))])
    mb = MV.voxelise(bridge, nx, ny, nz)
    assert mb[7, 7, 10] == 1 and mb[3, 7, 10] == 0 and mb[3, 7, 6] == 1
    o1.set_flags_mask(None, mb)
    fl = o1.get_flags()
    assert fl[7, 7, 10] == 1 and fl[3, 7, 10] == 0 and fl[0, 7, 10] == 0
    lk = o1.get_links()
    assert mb[6, 7, 10] == 1 and mb[5, 7, 10] == 0                            # slab = cells z 6..8 (centres 6.5 .. 8.5 in (6.4, 8.6))
    assert (lk[5, 7, 10] >> 5) & 1 == 0 and (lk[5, 7, 10] >> 6) & 1 == 1   # the cell under the slab pulls direction 6 = (0,0,-1) from the slab: bounce-back


def test_vertices_outside_the_allowed_range_are_refused(MV, W):
    with pytest.raises(ValueError):
        MV.voxelise(W.box_mesh((0, 0, 0), (3000, 2, 2)), 4, 4, 4)


# ---- the plain definition, cell by cell (DESIGN.md §4 reading 22) -----------------------------------------
# For every cell and every ray direction: count the triangles the ray through the cell centre crosses at or before the
# centre, with exact rational arithmetic.  No toggle array, no prefix sum, no floor division — none of the decomposition
# oracle/mesh_voxel.py (and the CUDA kernel) use — so a misconception shared by those two cannot pass here.

def plain_parities(MV, tri, nx, ny, nz):
    from fractions import Fraction as Fr
    v = [[[Fr(int(c), 256) for c in p] for p in t] for t in MV.snap(tri)]      # the snapped vertices, exact
    out = np.zeros((3, nz, ny, nx), dtype=np.uint8)
    for d in range(3):
        au, av, aw = (d + 1) % 3, (d + 2) % 3, d
        for z in range(nz):
            for y in range(ny):
                for x in range(nx):
                    ctr = (Fr(2 * x + 1, 2), Fr(2 * y + 1, 2), Fr(2 * z + 1, 2))
                    pu, pv, pw = ctr[au], ctr[av], ctr[aw]
                    crossings = 0
                    for a, b, c in v:
                        area = (b[au] - a[au]) * (c[av] - a[av]) - (b[av] - a[av]) * (c[au] - a[au])
                        if area == 0:
                            continue                                            # the ray lies in the triangle's plane
                        if area < 0:
                            b, c = c, b
                            area = -area                                        # counter-clockwise projection
                        lam = []
                        inside = True
                        for p, q in ((b, c), (c, a), (a, b)):                   # barycentric weight of a, b, c
                            du, dv = q[au] - p[au], q[av] - p[av]
                            e = du * (pv - p[av]) - dv * (pu - p[au])
                            if e < 0 or (e == 0 and not (dv < 0 or (dv == 0 and du > 0))):   # top-left rule on an edge
                                inside = False
                            lam.append(e / area)
                        if not inside:
                            continue
                        assert sum(lam) == 1
                        w_star = lam[0] * a[aw] + lam[1] * b[aw] + lam[2] * c[aw]
                        if w_star <= pw:                                        # crossing at or before the centre
                            crossings += 1
                    out[d, z, y, x] = crossings & 1
    return out[0], out[1], out[2]


def test_voxeliser_equals_the_plain_per_cell_definition_also_on_degenerate_meshes(MV, W):
    nx, ny, nz = 9, 8, 7
    rng = np.random.default_rng(12)
    meshes = {
        "corners on cell centres": W.box_mesh((1.5, 2.5, 1.5), (6.5, 5.5, 4.5)),
        "faces on cell faces": W.box_mesh((1.0, 2.0, 1.0), (6.0, 5.0, 4.0)),
        "two boxes sharing a face through centres": np.concatenate([W.box_mesh((1.25, 1.5, 0.75), (4.5, 6.25, 5.5)),
                                                                    W.box_mesh((4.5, 1.5, 0.75), (8.75, 6.25, 5.5))]),
        "clipped by the domain": W.box_mesh((-2.5, 3.5, -1.0), (4.5, 12.0, 3.5)),
        "sphere with a vertex column through centres": W.icosphere_mesh((4.5, 3.5, 3.5), 2.5, 1),
        "half a roof removed": np.delete(W.box_mesh((2.25, 2.25, 1.25), (7.75, 6.75, 5.75)), 10, axis=0),
    }
    # random triangles with vertices on the half-cell grid (every one of them degenerate for some ray), not closed
    meshes["random soup on the half-cell grid"] = (rng.integers(0, 16, size=(14, 3, 3)) / 2.0).astype(np.float32)
    meshes["random soup, generic"] = rng.uniform(-1, 9, size=(14, 3, 3)).astype(np.float32)
    for name, tri in meshes.items():
        want = plain_parities(MV, tri, nx, ny, nz)
        got = MV.pass_parities(tri, nx, ny, nz)
        for d in range(3):
            np.testing.assert_array_equal(got[d], want[d], err_msg=f"{name}, pass {d}")
        for votes in (1, 2, 3):
            np.testing.assert_array_equal(MV.voxelise(tri, nx, ny, nz, votes),
                                          ((want[0].astype(int) + want[1] + want[2]) >= votes).astype(np.uint8))
