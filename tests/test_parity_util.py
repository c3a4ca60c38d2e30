"""The two tie rules of the GPU parity checks are host logic on the oracle's fp64 geometry: pinned
here on rays built to have, or not to have, the tie, so that neither rule can accept an arbitrary ray.

Geometry of every case: a 4 x 4 x 4 volume of 2 mm voxels centred on the isocentre (lattice planes at -4, -2, 0, 2, 4 mm on
each axis), source at (-1000, 0, 0) (phi = 0), detector plane x = +500, u along +y, v along +z.  The ray to the pixel
at (u, v) is at y = u s, z = v s where s = (x + 1000) / 1500.
"""
import numpy as np

from parity_util import face_tie_checker, oracle_midpoints, siddon_sliver_checker
from test_oracle_pins import tiny_workload


def volume_with_marker(marker):
    rho = np.ones((4, 4, 4), dtype=np.float32)
    mat = np.zeros((4, 4, 4), dtype=np.uint8)
    ix, iy, iz = marker
    mat[iz, iy, ix] = 1
    return rho, mat


def test_sliver_tie_needs_two_planes_met_together_at_an_edge_of_the_material():
    # pixel column i = 3 of 5 at du = 3 mm: u = 3, so the ray meets the planes x = 0 (s = 2/3) and y = 2 in ONE point;
    # v = +0.75 (row 1 of 2 at dv = 1.5): z = 0.5 there, inside slab iz = 2, and z never reaches a plane inside the box.
    # The four voxels round that edge: ix in {1, 2}, iy in {2, 3}, iz = 2.
    kw = dict(n_materials=2, nu=5, nv=2, du=3.0, dv=1.5, phis=[0.0], mu_hat=np.full((2, 1), 0.02))
    tie_pixel, other_pixel = (0, 1, 1, 3), (0, 1, 1, 2)        # (projection, material, j, i); i = 2: u = 0, no y plane is met
    for marker in ((2, 2, 2), (1, 3, 2), (1, 2, 2), (2, 3, 2)):
        rho, mat = volume_with_marker(marker)
        w = tiny_workload(rho, mat, **kw)
        found = []
        check = siddon_sliver_checker(w, [0], found)
        assert check(tie_pixel), f"marker voxel {marker} is at the edge (x = 0, y = 2) the ray passes through"
        assert not check(other_pixel), "the ray in the plane y = 0 meets x planes only"
        assert found == [(0, 1, 1, 3), (0, 1, 1, 2)]
    # the material somewhere else: the tie is there, but it is not a tie of THIS material
    for marker in ((0, 0, 0), (2, 2, 0), (3, 2, 2), (1, 1, 2)):
        rho, mat = volume_with_marker(marker)
        w = tiny_workload(rho, mat, **kw)
        assert not siddon_sliver_checker(w, [0])(tie_pixel), f"marker voxel {marker} is not at the edge of the tie"
    # the material at the edge but empty (rho = 0): a sliver of it adds nothing, so it cannot explain a non-zero entry
    rho, mat = volume_with_marker((2, 2, 2))
    rho[2, 2, 2] = 0.0
    assert not siddon_sliver_checker(tiny_workload(rho, mat, **kw), [0])(tie_pixel)
    # an oblique ray (u = 2.2 at x = 500): its x and y crossings are 0.1 mm apart or more
    w = tiny_workload(*volume_with_marker((2, 2, 2)), n_materials=2, nu=5, nv=2, du=1.1, dv=1.5, phis=[0.0],
                      mu_hat=np.full((2, 1), 0.02))
    assert not siddon_sliver_checker(w, [0])((0, 1, 1, 4))


def test_face_tie_needs_a_midpoint_on_a_cell_face():
    rho = np.ones((4, 4, 4), dtype=np.float32)
    # the central ray (u = v = 0) runs along x from x = -4; midpoints at -4 + (k + 1/2) step.  step = 2/3 mm puts the
    # second midpoint at x = -3 = a voxel centre = a face of the tri-linear cells; step = 0.5 puts them at
    # -3.75, -3.25, ...: a quarter of a cell from every face.
    on_face = tiny_workload(rho, nu=3, nv=3, du=3.0, dv=3.0, phis=[0.0], step=2.0 / 3.0)
    off_face = tiny_workload(rho, nu=3, nv=3, du=3.0, dv=3.0, phis=[0.0], step=0.5)
    centre = (0, 0, 1, 1)
    assert face_tie_checker(on_face, [0])(centre)
    assert not face_tie_checker(off_face, [0])(centre)
    # a ray that misses the volume has no sample at all
    far = tiny_workload(rho, nu=3, nv=3, du=400.0, dv=400.0, phis=[0.0], step=0.5)
    assert not face_tie_checker(far, [0])((0, 0, 0, 0))
    assert not siddon_sliver_checker(far, [0])((0, 0, 0, 0))


def test_midpoints_rebuilt_from_the_ray_record_are_the_oracles():
    """oracle_midpoints (used by the face-tie rule, also for pose workloads) against oracle.ray_samples on the circular
    gantry, and the pose form against the circular form on the circle's own poses."""
    import oracle
    from workloads import trajectories
    rng = np.random.default_rng(4)
    rho = rng.uniform(0.0, 2.0, size=(9, 14, 11)).astype(np.float32)
    phis = np.radians([0.0, 33.0, 147.0, 301.5])
    w = tiny_workload(rho, spacing=(1.3, 0.9, 2.1), centre=(3.0, -2.0, 1.5), nu=21, nv=17, du=1.4, dv=1.7, phis=phis,
                      step=0.37, theta=0.004)
    wp = w.with_poses(trajectories.circular_poses(w.sad, w.sdd, w.theta, phis))
    seen = 0
    for p in range(len(phis)):
        for (i, j) in ((0, 0), (10, 8), (20, 16), (5, 12), (17, 3)):
            ref, _ = oracle.ray_samples(w, float(phis[p]), i, j)
            got = oracle_midpoints(w, p, i, j)
            assert got.shape == ref.shape
            if len(ref):
                assert np.abs(got - ref).max() < 1e-12
                assert np.abs(oracle_midpoints(wp, p, i, j) - ref).max() < 1e-9
                seen += len(ref)
    assert seen > 300
