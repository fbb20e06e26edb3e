"""GPU parity, stage by stage: libpmforce (fp32, through the C ABI binding) vs the fp64 oracle, element by
element on the same seeded inputs.  Meshes here span several tiles (8 x 8 x 16 cells) and ragged tails
(m = 40 is 2.5 tiles in z), particles span several work items.

Tolerances: scatter accumulates in 32-bit fixed point with a per-work-item
scale >= 2^19 / max|w| -> <= 1e-6 relative L2 on the mesh; gathers are fp32 FMAs -> <= 1e-6; the k-space
stage is fp32 cuFFT + fp64 symbols -> <= 2e-6.
"""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

from oracle import pm_oracle as po
from pm_inputs import generators as gen

from parity_util import MAXABS_SIGNED_SCATTER, check, record_error, rel_l2

pytestmark = pytest.mark.gpu


def _need_gpu():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")


@pytest.fixture(scope="module")
def pm():
    _need_gpu()
    import paper_2510_05206_b200 as pm_

    return pm_


def dev(x):
    return torch.from_numpy(np.ascontiguousarray(x)).cuda()


def mixed_positions(n, box, seed):
    """Uniform random + a dense clump (many particles in one tile -> several work items) + edge cases."""
    rng = np.random.default_rng(seed)
    a = gen.uniform_random(n, box, seed)
    clump = (rng.random((5000, 3)) * 0.02 + 0.31) * box
    edge = np.array([[0.0, 0.0, 0.0], [box * (1 - 2e-7), box * 0.5, 0.0], [box * 0.999999, box * 0.999999, box * 0.999999],
                     [-0.25 * box, 1.5 * box, 2.125 * box]])  # outside the box: wrapped periodically
    return np.concatenate([a, clump, edge]).astype(np.float32)


M = 40
BOX = 100.0


@pytest.mark.parametrize("worder", [2, 3, 4])
@pytest.mark.parametrize("shift_cells", [None, (0.5, 0.5, 0.5), (3.25, -1.5, 5.0)])
def test_assign_parity(pm, worder, shift_cells):
    pos = mixed_positions(30000, BOX, 11 + worder)
    shift = None if shift_cells is None else tuple(s * BOX / M for s in shift_cells)
    ctx = pm.pm_create(pm.PMParams(m=M, box=BOX, max_particles=pos.shape[0], worder=worder))
    mesh = torch.zeros(M, M, M, device="cuda")
    pm.pm_assign(ctx, dev(pos), None, mesh, shift=shift)
    ref = po.scatter(pos, M, BOX, worder, shift=shift)
    check("mesh", mesh, ref, 1e-6)
    # exact mass conservation (partition of unity), to fp32 accumulation
    assert abs(float(mesh.double().sum()) - pos.shape[0]) <= 1e-6 * pos.shape[0]
    # weighted, accumulating onto a pre-existing mesh
    w = np.random.default_rng(5).standard_normal(pos.shape[0]).astype(np.float32)
    pre = gen.random_mesh(M, 3)[0]
    mesh2 = dev(pre)
    pm.pm_assign(ctx, dev(pos), dev(w), mesh2, shift=shift)
    ref2 = po.scatter(pos, M, BOX, worder, weights=w, shift=shift, mesh=pre.astype(np.float64))
    check("mesh2", mesh2, ref2, 1e-6)
    pm.pm_destroy(ctx)


@pytest.mark.parametrize("worder", [2, 3, 4])
@pytest.mark.parametrize("shift_cells", [None, (0.5, 0.5, 0.5), (-2.75, 4.0, 0.125)])
@pytest.mark.parametrize("ncomp", [1, 2, 3])
def test_interp_parity(pm, worder, shift_cells, ncomp):
    pos = mixed_positions(20000, BOX, 21 + worder)
    shift = None if shift_cells is None else tuple(s * BOX / M for s in shift_cells)
    meshes = gen.random_mesh(M, 7, ncomp)
    ctx = pm.pm_create(pm.PMParams(m=M, box=BOX, max_particles=pos.shape[0], worder=worder))
    out = torch.empty(pos.shape[0], ncomp, device="cuda")
    pm.pm_interp(ctx, [dev(meshes[a]) for a in range(ncomp)], dev(pos), out, shift=shift)
    ref = np.stack([po.gather(meshes[a], pos, BOX, worder, shift=shift) for a in range(ncomp)], axis=1)
    check("out", out, ref, 1e-6)
    pm.pm_destroy(ctx)


@pytest.mark.parametrize("worder", [2, 3, 4])
@pytest.mark.parametrize("shifted", [False, True])
def test_assign_vjp_parity(pm, worder, shifted):
    pos = mixed_positions(20000, BOX, 31 + worder)
    n = pos.shape[0]
    shift = (0.5 * BOX / M,) * 3 if shifted else None
    w = np.random.default_rng(6).standard_normal(n).astype(np.float32)
    cot = gen.random_mesh(M, 8)[0]
    ctx = pm.pm_create(pm.PMParams(m=M, box=BOX, max_particles=n, worder=worder))
    pos_cot = torch.empty(n, 3, device="cuda")
    w_cot = torch.empty(n, device="cuda")
    pm.pm_assign_vjp(ctx, dev(pos), dev(w), dev(cot), pos_cot=pos_cot, w_cot=w_cot, shift=shift)
    ref_w = po.gather(cot, pos, BOX, worder, shift=shift)
    ref_p = np.stack([w * po.gather(cot, pos, BOX, worder, shift=shift, deriv_axis=b) for b in range(3)], axis=1)
    check("w_cot", w_cot, ref_w, 1e-6)
    check("pos_cot", pos_cot, ref_p, 2e-6)
    pm.pm_destroy(ctx)


@pytest.mark.parametrize("worder", [2, 3, 4])
@pytest.mark.parametrize("ncomp", [1, 3])
def test_interp_vjp_parity(pm, worder, ncomp):
    pos = mixed_positions(20000, BOX, 41 + worder)
    n = pos.shape[0]
    meshes = gen.random_mesh(M, 9, ncomp)
    cot = gen.gaussian_cotangent(n, 77, ncomp)
    ctx = pm.pm_create(pm.PMParams(m=M, box=BOX, max_particles=n, worder=worder))
    mesh_cot = [torch.zeros(M, M, M, device="cuda") for _ in range(ncomp)]
    pos_cot = torch.empty(n, 3, device="cuda")
    pm.pm_interp_vjp(ctx, [dev(meshes[a]) for a in range(ncomp)], dev(pos), dev(cot), mesh_cot=mesh_cot, pos_cot=pos_cot)
    for a in range(ncomp):
        ref = po.scatter(pos, M, BOX, worder, weights=cot[:, a])
        # random-sign weights in a dense clump: the node sums cancel, while the fixed-point quantum is 2^-30 of the
        # work item's bound sum|w| * Wmax^3 ("Parity bars"); with items of up to 4096 particles that is
        # the accuracy of an fp32 accumulation in the same order, not better
        check("mesh_cot[a]", mesh_cot[a], ref, 5e-6, maxabs_tol=MAXABS_SIGNED_SCATTER)
    ref_p = np.zeros((n, 3))
    for a in range(ncomp):
        for b in range(3):
            ref_p[:, b] += cot[:, a] * po.gather(meshes[a], pos, BOX, worder, deriv_axis=b)
    check("pos_cot", pos_cot, ref_p, 2e-6)
    pm.pm_destroy(ctx)


def test_adjointness_on_gpu(pm):
    """<gather(f), w> = <f, scatter(w)>  (Eq. C.14) with the GPU operators."""
    pos = mixed_positions(20000, BOX, 51)
    n = pos.shape[0]
    w = np.random.default_rng(8).standard_normal(n).astype(np.float32)
    f = gen.random_mesh(M, 10)[0]
    for worder in (2, 3, 4):
        ctx = pm.pm_create(pm.PMParams(m=M, box=BOX, max_particles=n, worder=worder))
        mesh = torch.zeros(M, M, M, device="cuda")
        pm.pm_assign(ctx, dev(pos), dev(w), mesh)
        out = torch.empty(n, 1, device="cuda")
        pm.pm_interp(ctx, [dev(f)], dev(pos), out)
        lhs = float((out[:, 0].double() * dev(w).double()).sum())
        rhs = float((mesh.double() * dev(f).double()).sum())
        scale = float(np.sqrt(n)) * 1.0
        assert abs(lhs - rhs) <= 2e-5 * scale
        pm.pm_destroy(ctx)


@pytest.mark.parametrize("grad_order,lap_order,deconv_pow,worder", [
    (0, 0, 2, 2), (2, 2, 0, 2), (4, 0, 2, 3), (6, 6, 1, 4), (4, 4, 0, 2), (0, 6, 2, 3)])
def test_poisson_force_parity(pm, grad_order, lap_order, deconv_pow, worder):
    m, box = 32, 64.0
    delta = gen.random_mesh(m, 12)[0]
    ctx = pm.pm_create(pm.PMParams(m=m, box=box, max_particles=8, worder=worder, grad_order=grad_order,
                                   lap_order=lap_order, deconv_pow=deconv_pow, coeff=1.7))
    g = [torch.empty(m, m, m, device="cuda") for _ in range(3)]
    pm.pm_poisson_force(ctx, dev(delta), g)
    ref = po.poisson_force(delta, box, worder, grad_order, lap_order, deconv_pow, coeff=1.7)
    for a in range(3):
        check("g[a]", g[a], ref[a], 2e-6)
    # transpose
    cot = gen.random_mesh(m, 13, 3)
    dc = torch.empty(m, m, m, device="cuda")
    pm.pm_poisson_force_vjp(ctx, [dev(cot[a]) for a in range(3)], dc)
    refv = po.poisson_force_vjp([cot[a] for a in range(3)], box, worder, grad_order, lap_order, deconv_pow, coeff=1.7)
    check("dc", dc, refv, 2e-6)
    pm.pm_destroy(ctx)


def test_poisson_force_interlaced_parity(pm):
    m, box = 32, 64.0
    d = gen.random_mesh(m, 14, 2)
    ctx = pm.pm_create(pm.PMParams(m=m, box=box, max_particles=8, worder=3, grad_order=4, interlace=1))
    g = [torch.empty(m, m, m, device="cuda") for _ in range(3)]
    pm.pm_poisson_force(ctx, dev(d[0]), g, delta_mesh2=dev(d[1]))
    ref = po.poisson_force(d[0], box, 3, 4, 0, 2, delta_mesh2=d[1])
    for a in range(3):
        check("g[a]", g[a], ref[a], 2e-6)
    cot = gen.random_mesh(m, 15, 3)
    c1 = torch.empty(m, m, m, device="cuda")
    c2 = torch.empty(m, m, m, device="cuda")
    pm.pm_poisson_force_vjp(ctx, [dev(cot[a]) for a in range(3)], c1, delta_cot2=c2)
    r1, r2 = po.poisson_force_vjp([cot[a] for a in range(3)], box, 3, 4, 0, 2, interlace=True)
    check("c1", c1, r1, 2e-6)
    check("c2", c2, r2, 2e-6)
    pm.pm_destroy(ctx)


def test_edge_cases(pm):
    """N = 1; all particles in one cell (many work items, heavy atomic contention); smallest mesh."""
    # one particle
    ctx = pm.pm_create(pm.PMParams(m=8, box=8.0, max_particles=20000, worder=4))
    p1 = np.array([[7.9, 0.05, 3.5]], dtype=np.float32)
    mesh = torch.zeros(8, 8, 8, device="cuda")
    pm.pm_assign(ctx, dev(p1), None, mesh)
    check("one_particle", mesh, po.scatter(p1, 8, 8.0, 4), 1e-6)
    # 20000 particles inside one cell of an 8^3 mesh whose kernel support wraps around the box
    rng = np.random.default_rng(3)
    pc = (rng.random((20000, 3)) * 0.9 + np.array([7.05, 0.05, 7.05])).astype(np.float32) % np.float32(8.0)
    mesh.zero_()
    pm.pm_assign(ctx, dev(pc), None, mesh)
    check("one_cell", mesh, po.scatter(pc, 8, 8.0, 4), 1e-6)
    f = gen.random_mesh(8, 4, 3)
    out = torch.empty(20000, 3, device="cuda")
    pm.pm_interp(ctx, [dev(f[a]) for a in range(3)], dev(pc), out)
    ref = np.stack([po.gather(f[a], pc, 8.0, 4) for a in range(3)], axis=1)
    check("out", out, ref, 1e-6)
    pm.pm_destroy(ctx)


def test_bucket_overflow_of_single_pass_binning(pm):
    """Half of the particles inside two tiles of a 64^3 mesh (128 tiles, bucket = twice the mean load): their
    records overflow the tile buckets and take the overflow-sort path of the binning; assign and interp must
    still match the oracle, and the forces must come back in caller order."""
    m, box, n = 64, 64.0, 60000
    rng = np.random.default_rng(11)
    pu = rng.random((n // 2, 3)) * box
    pa = rng.random((n // 4, 3)) * np.array([7.9, 7.9, 31.9]) + np.array([8.0, 16.0, 32.0])
    pb = rng.random((n - n // 2 - n // 4, 3)) * np.array([7.9, 7.9, 31.9]) + np.array([56.0, 56.0, 0.0])
    pos = np.concatenate([pu, pa, pb]).astype(np.float32)
    pos = pos[rng.permutation(n)]
    for worder in (2, 3):
        ctx = pm.pm_create(pm.PMParams(m=m, box=box, max_particles=n, worder=worder))
        mesh = torch.zeros(m, m, m, device="cuda")
        pm.pm_assign(ctx, dev(pos), None, mesh)
        ref = po.scatter(pos, m, box, worder)
        check("mesh", mesh, ref, 1e-6)
        assert abs(float(mesh.sum().cpu()) - n) <= 1e-4 * n
        f = gen.random_mesh(m, 5, 3)
        out = torch.empty(n, 3, device="cuda")
        pm.pm_interp(ctx, [dev(f[a]) for a in range(3)], dev(pos), out)
        refg = np.stack([po.gather(f[a], pos, box, worder) for a in range(3)], axis=1)
        check("out", out, refg, 1e-6)
        pm.pm_destroy(ctx)


def test_two_pass_binning_path_matches(pm):
    """The two-pass (histogram + permute) binning, kept for N too large for 32-bit bucket indices and selectable
    with PM_FLAG_BIN_TWOPASS, must give the same assignment and forces as the default single-pass path."""
    pos, c = gen.make_config_positions("cfg4", n_p=32)
    n = pos.shape[0]
    f = gen.random_mesh(c["m"], 6, 3)
    ref = po.scatter(pos, c["m"], c["box"], 2)
    outs = []
    for flags in (0, pm.FLAG_BIN_TWOPASS):
        ctx = pm.pm_create(pm.PMParams(m=c["m"], box=c["box"], max_particles=n, worder=2, flags=flags))
        mesh = torch.zeros(c["m"], c["m"], c["m"], device="cuda")
        pm.pm_assign(ctx, dev(pos), None, mesh)
        out = torch.empty(n, 3, device="cuda")
        pm.pm_interp(ctx, [dev(f[a]) for a in range(3)], dev(pos), out)
        check("mesh", mesh, ref, 1e-6)
        outs.append(out.cpu().numpy())
        pm.pm_destroy(ctx)
    # the gather of one particle does not depend on how the records were sorted
    assert np.array_equal(outs[0], outs[1])


def test_errors_are_reported(pm):
    with pytest.raises(pm.PMError):
        pm.pm_create(pm.PMParams(m=30, box=1.0, max_particles=10))  # m not a multiple of 4
    ctx = pm.pm_create(pm.PMParams(m=16, box=1.0, max_particles=10))
    pos = torch.zeros(11, 3, device="cuda")
    with pytest.raises(pm.PMError):
        pm.pm_bin(ctx, pos)  # N > max_particles
    with pytest.raises(pm.PMError):
        pm.nufft_spread(ctx, pos[:4], None, torch.zeros(16, 16, 16, device="cuda"))  # PM ctx
    pm.pm_destroy(ctx)


def test_pm_bin_pinned_records_are_reused(pm):
    """pm_bin pins the sorted records: pm_assign, pm_interp, pm_interp_vjp and pm_assign_vjp given the same
    (pos, N) reuse them (include/pmforce.h); results must equal the calls that bin internally, and a call with
    other positions must drop the pin and bin again."""
    pos = mixed_positions(20000, BOX, 91)
    n = pos.shape[0]
    d_pos = dev(pos)
    meshes = gen.random_mesh(M, 92, 3)
    d_m = [dev(meshes[a]) for a in range(3)]
    cot = gen.gaussian_cotangent(n, 93, 3)
    for worder in (2, 3):
        ctx = pm.pm_create(pm.PMParams(m=M, box=BOX, max_particles=n, worder=worder))
        pm.pm_bin(ctx, d_pos)
        mesh = torch.zeros(M, M, M, device="cuda")
        pm.pm_assign(ctx, d_pos, None, mesh)
        check("pinned/assign", mesh, po.scatter(pos, M, BOX, worder), 1e-6)
        out = torch.empty(n, 3, device="cuda")
        pm.pm_interp(ctx, d_m, d_pos, out)
        ref = np.stack([po.gather(meshes[a], pos, BOX, worder) for a in range(3)], axis=1)
        check("pinned/interp", out, ref, 1e-6)
        pc = torch.empty(n, 3, device="cuda")
        mc = [torch.zeros(M, M, M, device="cuda") for _ in range(3)]
        pm.pm_interp_vjp(ctx, d_m, d_pos, dev(cot), mesh_cot=mc, pos_cot=pc)
        refp = np.zeros((n, 3))
        for a in range(3):
            check(f"pinned/mesh_cot{a}", mc[a], po.scatter(pos, M, BOX, worder, weights=cot[:, a]), 5e-6,
                  maxabs_tol=MAXABS_SIGNED_SCATTER)
            for b in range(3):
                refp[:, b] += cot[:, a] * po.gather(meshes[a], pos, BOX, worder, deriv_axis=b)
        check("pinned/pos_cot", pc, refp, 2e-6)
        # other positions at another address: the pin is dropped, the records are rebuilt
        pos2 = mixed_positions(20000, BOX, 94)
        out2 = torch.empty(n, 3, device="cuda")
        pm.pm_interp(ctx, d_m, dev(pos2), out2)
        ref2 = np.stack([po.gather(meshes[a], pos2, BOX, worder) for a in range(3)], axis=1)
        check("repinned/interp", out2, ref2, 1e-6)
        pm.pm_destroy(ctx)
