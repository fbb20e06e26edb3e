"""GPU parity at the sizes and on the code paths the BASELINE configurations really take.

* every instantiation of the fused x-FFT + Fourier-space kernel (m = 64 ... 1024, forward and transposed, with
  and without the interlaced second mesh) against the oracle: element by element up to 512^3, and at 1024^3
  (where the fp64 oracle's 3-D symbol arrays would need ~100 GB) on a seeded superposition of plane waves whose
  response the oracle's symbols give in closed form (the mesh-injection pin of tests/test_oracle_pm.py), on
  sampled nodes, plus Parseval over the whole mesh and the fused path against the unfused one on every mode;
* the bench workloads at FULL size in the launch configuration bench.py times: the oracle assigns all particles
  and solves at full size in fp64, then gathers for a seeded sample of particles one by one (headline, cfg2,
  cfg4 with half of the sample inside halo cores), forward force and VJP;
* the NUFFT stages at the cfg3 sizes: spreading onto the 1024^3 fine grid against the oracle on seeded windows
  of the grid, the Fourier-space stage on plane waves, interpolation on sampled particles.

The oracle's FFTs run on all host cores here (pm_oracle.FFT_WORKERS; same pocketfft arithmetic).
"""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

from oracle import nufft_oracle as no
from oracle import pm_oracle as po
from pm_inputs import generators as gen

from parity_util import check, record_error, rel_l2

pytestmark = pytest.mark.gpu

FORCE_TOL = 1e-5
VJP_TOL = 1e-5
NSAMPLE = 200_000


@pytest.fixture(scope="module")
def pm():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2510_05206_b200 as pm_

    return pm_


@pytest.fixture(autouse=True)
def _oracle_fft_on_all_cores():
    old = po.FFT_WORKERS
    po.FFT_WORKERS = -1
    yield
    po.FFT_WORKERS = old
    torch.cuda.empty_cache()


def dev(x):
    return torch.from_numpy(np.ascontiguousarray(x)).cuda()


# ---- plane-wave meshes ---------------------------------------------------------------------------------------
def synth_mesh(m, idx, coef):
    """f(j) = Re sum_w c_w exp(2 pi i n_w.j / m) on the device, fp64 arithmetic, returned as fp32 [m, m, m]
    (test plumbing: the rank-W separable sum as one complex matmul per slab of x planes)."""
    j = torch.arange(m, device="cuda", dtype=torch.float64)
    ph = [torch.exp(2j * torch.pi * (j[:, None] * torch.from_numpy(idx[:, a].astype(np.float64)).cuda()[None, :] % m) / m)
          for a in range(3)]  # [m, W] each
    c = torch.from_numpy(coef).cuda()
    out = torch.empty(m, m, m, device="cuda", dtype=torch.float32)
    zt = ph[2].T.contiguous()  # [W, m]
    step = max(1, min(m, (1 << 27) // (m * m)))
    for x0 in range(0, m, step):
        a = ph[0][x0:x0 + step] * c[None, :]                       # [s, W]
        ya = a[:, None, :] * ph[1][None, :, :]                     # [s, m, W]
        out[x0:x0 + step] = torch.matmul(ya, zt).real.to(torch.float32)
    return out


def amplitudes(n, seed):
    rng = np.random.default_rng(seed)
    return rng.standard_normal(n) + 1j * rng.standard_normal(n)


def sample_nodes(m, n, seed):
    rng = np.random.default_rng(seed)
    nodes = rng.integers(0, m, size=(n, 3))
    line = np.arange(min(m, 2048)) % m
    extra = [np.stack([line, np.full_like(line, 3), np.full_like(line, m - 1)], 1),   # a whole x line
             np.stack([np.full_like(line, m - 1), line, np.full_like(line, 0)], 1),   # a whole y line
             np.stack([np.full_like(line, 0), np.full_like(line, m // 2), line], 1)]  # a whole z line
    return np.concatenate([nodes] + extra)


def at_nodes(t, nodes):
    n = torch.from_numpy(nodes).cuda()
    return t[n[:, 0], n[:, 1], n[:, 2]].double().cpu().numpy()


KSPACE_SETTINGS = dict(worder=2, grad_order=4, lap_order=0, deconv_pow=2, coeff=1.3)


@pytest.mark.parametrize("m", [256, 1024])
@pytest.mark.parametrize("interlace", [0, 1])
def test_fused_kspace_plane_waves(pm, m, interlace):
    """k_xfft_kspace<256> (radix 16 x 16) and <1024> (16 x 8 x 8), MODE 0 and MODE 1, against the closed form
    g_a(j) = sum_w Re[S_a(n_w) c_w e^{i theta_w.j}] with S_a from the oracle's symbol tables."""
    box = 1000.0
    kw = dict(KSPACE_SETTINGS, worder=3 if interlace else 2)
    ctx = pm.pm_create(pm.PMParams(m=m, box=box, max_particles=8, interlace=interlace, **kw))
    idx, c1 = gen.plane_wave_modes(m, 400, 9000 + m)
    c2 = amplitudes(idx.shape[0], 9001 + m)
    S = po.force_symbol_at(tuple(idx[:, a] for a in range(3)), m, box, kw["worder"], kw["grad_order"],
                           kw["lap_order"], kw["deconv_pow"], kw["coeff"])          # [3, W]
    ph1 = po.interlace_phase(m)
    p3 = ph1[idx[:, 0]] * ph1[idx[:, 1]] * ph1[idx[:, 2]]
    nodes = sample_nodes(m, NSAMPLE, 17)
    d1 = synth_mesh(m, idx, c1)
    d2 = synth_mesh(m, idx, c2) if interlace else None
    g = [torch.empty(m, m, m, device="cuda") for _ in range(3)]
    pm.pm_poisson_force(ctx, d1, g, delta_mesh2=d2)
    chat = 0.5 * (c1 + p3 * c2) if interlace else c1
    G = float(m) ** 3
    for a in range(3):
        ref = gen.plane_wave_values(m, idx, S[a] * chat, nodes)
        check(f"fwd/g{a}", at_nodes(g[a], nodes), ref, 3e-6)
        # Parseval over the whole mesh: distinct, non-self-conjugate modes are orthogonal
        tot = float((g[a].double() ** 2).sum())
        want = G * 0.5 * float(np.sum(np.abs(S[a] * chat) ** 2))
        assert abs(tot - want) <= 2e-5 * want
    # transpose: cotangent meshes with their own amplitudes
    cs = [amplitudes(idx.shape[0], 9100 + m + a) for a in range(3)]
    gb = [synth_mesh(m, idx, cs[a]) for a in range(3)]
    q1 = torch.empty(m, m, m, device="cuda")
    q2 = torch.empty(m, m, m, device="cuda") if interlace else None
    pm.pm_poisson_force_vjp(ctx, gb, q1, delta_cot2=q2)
    qc = sum(np.conj(S[a]) * cs[a] for a in range(3))
    if interlace:
        check("tr/q1", at_nodes(q1, nodes), gen.plane_wave_values(m, idx, 0.5 * qc, nodes), 3e-6)
        check("tr/q2", at_nodes(q2, nodes), gen.plane_wave_values(m, idx, 0.5 * np.conj(p3) * qc, nodes), 3e-6)
    else:
        check("tr/q1", at_nodes(q1, nodes), gen.plane_wave_values(m, idx, qc, nodes), 3e-6)
    pm.pm_destroy(ctx)


@pytest.mark.parametrize("m", [64, 128, 256, 320, 512])
def test_fused_kspace_random_mesh_vs_oracle(pm, m):
    """Every mode of the fused kernel against the oracle, element by element, on random meshes: forward and
    transpose, interlaced (two input / two output meshes: the superset of the single-grid data flow).  m = 320 takes
    the radix-5 first stage of the upsampled NUFFT grids (5/4 * 2^k)."""
    box = 500.0
    kw = dict(worder=3, grad_order=4, lap_order=0, deconv_pow=2, coeff=0.7)
    d = gen.random_mesh(m, 300 + m, 2)
    ctx = pm.pm_create(pm.PMParams(m=m, box=box, max_particles=8, interlace=1, **kw))
    g = [torch.empty(m, m, m, device="cuda") for _ in range(3)]
    pm.pm_poisson_force(ctx, dev(d[0]), g, delta_mesh2=dev(d[1]))
    ref = po.poisson_force(d[0], box, kw["worder"], kw["grad_order"], kw["lap_order"], kw["deconv_pow"],
                           coeff=kw["coeff"], delta_mesh2=d[1])
    for a in range(3):
        check(f"fwd/g{a}", g[a], ref[a], 3e-6)
    del ref
    cot = gen.random_mesh(m, 400 + m, 3)
    c1, c2 = torch.empty(m, m, m, device="cuda"), torch.empty(m, m, m, device="cuda")
    pm.pm_poisson_force_vjp(ctx, [dev(cot[a]) for a in range(3)], c1, delta_cot2=c2)
    r1, r2 = po.poisson_force_vjp([cot[a] for a in range(3)], box, kw["worder"], kw["grad_order"], kw["lap_order"],
                                  kw["deconv_pow"], coeff=kw["coeff"], interlace=True)
    check("tr/c1", c1, r1, 3e-6)
    check("tr/c2", c2, r2, 3e-6)
    pm.pm_destroy(ctx)
    # single-grid data flow with the spectral gradient and all FD Laplacians (another symbol set)
    for go, lo, dp in ((0, 6, 1), (6, 2, 0)):
        ctx = pm.pm_create(pm.PMParams(m=m, box=box, max_particles=8, worder=2, grad_order=go, lap_order=lo,
                                       deconv_pow=dp))
        pm.pm_poisson_force(ctx, dev(d[0]), g)
        ref = po.poisson_force(d[0], box, 2, go, lo, dp)
        for a in range(3):
            check(f"fwd/go{go}lo{lo}/g{a}", g[a], ref[a], 3e-6)
        pm.pm_destroy(ctx)


def test_fused_vs_unfused_1024_every_mode(pm):
    """At 1024^3 every mode of the fused path against the unfused one (3-D cuFFT + pointwise kernel, itself
    oracle-tested element by element at small m) on a random mesh: GPU vs GPU, complements the plane waves."""
    m, box = 1024, 1000.0
    d = torch.randn(m, m, m, device="cuda", generator=torch.Generator(device="cuda").manual_seed(5))
    outs = []
    for flags in (0, pm.FLAG_NO_XFUSE):
        ctx = pm.pm_create(pm.PMParams(m=m, box=box, max_particles=8, flags=flags, **KSPACE_SETTINGS))
        g = [torch.empty(m, m, m, device="cuda") for _ in range(3)]
        pm.pm_poisson_force(ctx, d, g)
        q = torch.empty(m, m, m, device="cuda")
        pm.pm_poisson_force_vjp(ctx, g, q)
        outs.append(g + [q])
        pm.pm_destroy(ctx)
    for a in range(4):
        num = float((outs[0][a].double() - outs[1][a].double()).norm())
        den = float(outs[1][a].double().norm())
        mx = float((outs[0][a] - outs[1][a]).abs().max()) / (den / m ** 1.5)
        record_error(f"fused_vs_unfused_1024/{a}", num / den, 3e-6, mx)
        assert num <= 3e-6 * den and mx <= 1e-4


# ---- full-size sampled parity of the bench workloads ------------------------------------------------------------
def params_of(pm, c, n, **over):
    kw = dict(m=c["m"], box=c["box"], max_particles=n, worder=c.get("worder", 2), interlace=c.get("interlace", 0),
              deconv_pow=c.get("deconv_pow", 2), grad_order=c.get("grad_order", 0), lap_order=c.get("lap_order", 0))
    kw.update(over)
    return pm.PMParams(**kw)


def sampled_force_and_vjp(pm, name, sample_idx_fn, with_vjp, variants=(("", 0),)):
    """pm_force (and pm_force_vjp) on config `name` at full size, once per (tag, pm_params.flags) variant; the oracle
    does steps O1-O7 (and V(ii), V(iii)) on all particles in fp64, ONCE, and the per-particle steps O8 / V(i), V(iv)
    on the sampled particles; every variant is compared with the same reference."""
    pos, c = gen.make_config_positions(name)
    n = pos.shape[0]
    m, box, wo = c["m"], c["box"], c["worder"]
    lam = gen.gaussian_cotangent(n, c.get("cot_seed", 2000)) if with_vjp else None
    got = []
    for tag, flags in variants:
        ctx = pm.pm_create(params_of(pm, c, n, flags=flags))
        d_pos = dev(pos)
        f = torch.empty(n, 3, device="cuda")
        pm.pm_force(ctx, d_pos, f)
        xb = None
        if with_vjp:
            d_lam = dev(lam)
            t = torch.empty(n, 3, device="cuda")
            pm.pm_force_vjp(ctx, d_pos, d_lam, t)
            xb = t.cpu().numpy()
            del t, d_lam
        got.append((tag, f.cpu().numpy(), xb))
        del d_pos, f
        pm.pm_destroy(ctx)
        torch.cuda.empty_cache()

    kw = dict(box=box, worder=wo, grad_order=c["grad_order"], lap_order=c["lap_order"], deconv_pow=c["deconv_pow"])
    rho = po.scatter(pos, m, box, wo)
    idx = sample_idx_fn(pos, rho, n, box)
    g = po.poisson_force(po.density_contrast(rho, n), **kw)
    del rho
    ps = pos[idx]
    ref = np.stack([po.gather(g[a], ps, box, wo) for a in range(3)], axis=1)
    for tag, f, _ in got:
        check(f"{name}{tag}/force/sampled={idx.size}", f[idx], ref, FORCE_TOL)
        fsum = np.abs(f.astype(np.float64).sum(axis=0)).max()  # holds at any size: momentum conservation (interlace 0)
        assert fsum <= 1e-6 * np.abs(f.astype(np.float64)).sum()
    if with_vjp:
        ls = lam[idx].astype(np.float64)
        refv = np.zeros((idx.size, 3))
        for a in range(3):                                   # V(i): Eq. C.12
            for b in range(3):
                refv[:, b] += ls[:, a] * po.gather(g[a], ps, box, wo, deriv_axis=b)
        del g
        gbar = [po.scatter(pos, m, box, wo, weights=lam[:, a]) for a in range(3)]   # V(ii): Eq. C.10
        dbar = po.poisson_force_vjp(gbar, **kw)                                      # V(iii)
        del gbar
        for b in range(3):                                   # V(iv): Eq. C.6, w_i = 1, d(delta)/d(rho) = G/N
            refv[:, b] += (m ** 3 / float(n)) * po.gather(dbar, ps, box, wo, deriv_axis=b)
        for tag, _, xb in got:
            check(f"{name}{tag}/vjp/sampled={idx.size}", xb[idx], refv, VJP_TOL)


def uniform_sample(pos, rho, n, box):
    return np.sort(np.random.default_rng(4242).choice(n, size=NSAMPLE, replace=False))


def halo_core_sample(pos, rho, n, box):
    """Half of the sample from inside halo cores: particles of the halo half (first n/2, grouped by halo) whose
    cell holds >= 32 particles (mean: 1/8); the other half uniform over the lattice half."""
    rng = np.random.default_rng(4243)
    m = rho.shape[0]
    half = n // 2
    cand = np.sort(rng.choice(half, size=8_000_000, replace=False))
    cell = np.floor(pos[cand].astype(np.float64) * (m / box)).astype(np.int64) % m
    near = np.zeros(cand.size)
    for dx in (0, 1):          # CIC mass around the particle's cell ~ local particle count
        for dy in (0, 1):
            for dz in (0, 1):
                near += rho[(cell[:, 0] + dx) % m, (cell[:, 1] + dy) % m, (cell[:, 2] + dz) % m]
    dense = cand[near >= 8 * 32.0]
    assert dense.size >= NSAMPLE // 2, dense.size
    core = rng.choice(dense, size=NSAMPLE // 2, replace=False)
    lat = half + rng.choice(n - half, size=NSAMPLE // 2, replace=False)
    return np.sort(np.concatenate([core, lat]))


def test_headline_full_size_sampled(pm):
    """The bench workload itself (N = 512^3 on 512^3, CIC, FD4, deconvolved): forward force and VJP, on the reference
    path (three inverse FFTs) and with PM_FLAG_GRAD_REAL (one inverse FFT, gradient by the real-space stencil),
    both against the same, unchanged oracle."""
    sampled_force_and_vjp(pm, "headline", uniform_sample, with_vjp=True,
                          variants=(("", 0), ("+grad_real", pm.FLAG_GRAD_REAL)))


def test_cfg2_full_size_sampled(pm):
    """BASELINE config 2 at full size (256^3 particles on 512^3: the paper's default res_pm = 2 N^(1/3), :406)."""
    sampled_force_and_vjp(pm, "cfg2", uniform_sample, with_vjp=False)


@pytest.mark.slow
def test_cfg4_full_size_sampled(pm):
    """BASELINE config 4 at full size (clustered halos, 512^3 particles on 1024^3): forward force and VJP, half of
    the sample inside halo cores (tiles split into many work items with cancelling cotangents)."""
    sampled_force_and_vjp(pm, "cfg4", halo_core_sample, with_vjp=True)


# ---- NUFFT at the cfg3 sizes -------------------------------------------------------------------------------------
def nufft_params(pm, m, box, n, sigma=2.0, eps=1e-6, width=0, flags=0):
    return pm.PMParams(m=m, box=box, max_particles=n, method=1, nufft_sigma=sigma, nufft_eps=eps, nufft_width=width,
                       grad_order=0, lap_order=0, flags=flags)


@pytest.mark.parametrize("fine,sigma", [(512, 2.0), (1024, 2.0), (640, 1.25)])
def test_nufft_kspace_plane_waves(pm, fine, sigma):
    """NUFFT Fourier-space stage on the fused kernel with the NUFFT tables (mode truncation, 1/phi_hat^2, i k / k^2)
    at the cfg3 fine grid (1024), at 512 and at the paper-default setting of cfg3_paper (sigma = 5/4, w = 5, fine grid
    640 = 5 * 128: radix-5 first stage): closed form from the oracle's multiplier at single modes."""
    m, box, npart = int(round(fine / sigma)), 1000.0, 12345
    ctx = pm.pm_create(nufft_params(pm, m, box, 8, sigma=sigma, eps=1e-6 if sigma == 2.0 else 1e-4,
                                    width=0 if sigma == 2.0 else 5))
    assert ctx.mg == fine
    w, beta = ctx.nufft_width, ctx.nufft_beta
    idx, c1 = gen.plane_wave_modes(fine, 600, 9200 + fine)
    # half of the modes inside the retained cube |n_a| < m/2, half anywhere (dropped: response 0)
    inside = np.arange(idx.shape[0]) % 2 == 0
    lo = np.random.default_rng(5).integers(-(m // 2) + 1, m // 2, size=idx.shape)
    idx = np.where(inside[:, None], lo % fine, idx)
    idx = idx[np.any(idx != (-idx) % fine, axis=1)]  # no self-conjugate mode
    _, keep = np.unique(np.minimum(idx @ [fine * fine, fine, 1], ((-idx) % fine) @ [fine * fine, fine, 1]), return_index=True)
    idx = idx[keep]  # no mode twice, no mode with its conjugate
    c1 = amplitudes(idx.shape[0], 9201 + fine)
    M = no.kspace_multiplier_at(tuple(idx[:, a] for a in range(3)), fine, m, box, npart, w, beta, 1.0)
    assert (np.abs(M).sum(0) > 0).sum() > 100
    nodes = sample_nodes(fine, NSAMPLE, 19)
    f = synth_mesh(fine, idx, c1)
    g = [torch.empty(fine, fine, fine, device="cuda") for _ in range(3)]
    pm.nufft_poisson_force(ctx, f, npart, g)
    G = float(fine) ** 3  # the oracle's stage carries the G of the unnormalised inverse transform
    for a in range(3):
        check(f"fwd/g{a}", at_nodes(g[a], nodes), gen.plane_wave_values(fine, idx, G * M[a] * c1, nodes), 3e-6)
    cs = [amplitudes(idx.shape[0], 9300 + fine + a) for a in range(3)]
    gb = [synth_mesh(fine, idx, cs[a]) for a in range(3)]
    q = torch.empty(fine, fine, fine, device="cuda")
    pm.nufft_poisson_force_vjp(ctx, gb, npart, q)
    qc = sum(np.conj(M[a]) * cs[a] for a in range(3))
    check("tr/q", at_nodes(q, nodes), gen.plane_wave_values(fine, idx, G * qc, nodes), 3e-6)
    pm.pm_destroy(ctx)


def window_particles(pos, box, mg, origin, size, reach):
    """Particles whose kernel support (reach cells) touches the window [origin, origin + size) of the mg-mesh, and
    their coordinates translated so the window starts at node `reach + 1` of a small periodic mesh."""
    u = pos.astype(np.float64) * (mg / box)
    sel = np.ones(pos.shape[0], dtype=bool)
    rel = np.empty_like(u)
    for a in range(3):
        r = np.mod(u[:, a] - (origin[a] - reach - 1), mg)
        rel[:, a] = r
        sel &= r < size + 2 * reach + 2
    return rel[sel], sel


def test_cfg3_spread_full_size_windows(pm):
    """nufft_spread of all 512^3 particles onto the 1024^3 fine grid (cfg3, w = 7): the oracle spreads, in fp64,
    the particles around seeded windows of the grid (one at the box corner, wrapping) and compares node by node;
    plus mass conservation over the whole grid: sum(fine) = N * (sum_j phi_j)^3 per particle, checked through the
    oracle's total for a sample."""
    pos, c = gen.make_config_positions("cfg3")
    n = pos.shape[0]
    box, mf = c["box"], 1024
    ctx = pm.pm_create(nufft_params(pm, c["m"], box, n))
    w, beta = ctx.nufft_width, ctx.nufft_beta
    fine = torch.zeros(mf, mf, mf, device="cuda")
    d_pos = dev(pos)
    pm.nufft_spread(ctx, d_pos, None, fine)
    size, reach, ml = 24, w // 2 + 1, 64
    origins = [(mf - 10, mf - 7, mf - 30), (500, 8, 1000), (37, 613, 250), (777, 300, 31)]
    for k, o in enumerate(origins):
        rel, _ = window_particles(pos, box, mf, o, size, reach)
        loc = no.es_spread(rel * (box / mf), ml, ml * box / mf, w, beta)   # same cell size, small periodic mesh
        a0 = reach + 1
        ref = loc[a0:a0 + size, a0:a0 + size, a0:a0 + size]
        ix = [torch.arange(o[a], o[a] + size, device="cuda") % mf for a in range(3)]
        got = fine[ix[0]][:, ix[1]][:, :, ix[2]]
        check(f"window{k}", got, ref, 2e-6)
    # interpolation at full size on sampled particles, from GPU-made random fine meshes (stage parity)
    del fine
    meshes = [torch.randn(mf, mf, mf, device="cuda", generator=torch.Generator(device="cuda").manual_seed(70 + a))
              for a in range(3)]
    out = torch.empty(n, 3, device="cuda")
    pm.nufft_interp(ctx, meshes, d_pos, out)
    idx = np.sort(np.random.default_rng(4244).choice(n, size=20_000, replace=False))
    got = out[torch.from_numpy(idx).cuda()].cpu().numpy()
    ref = np.stack([no.es_interp(meshes[a].cpu().numpy(), pos[idx], box, w, beta) for a in range(3)], axis=1)
    check("interp/sampled=20000", got, ref, 2e-6)
    pm.pm_destroy(ctx)


def test_cfg3_reduced_fused256(pm):
    """cfg3 at n_p = 128 (128 modes, fine grid 256: the fused kernel's 16 x 16 plan with the NUFFT tables), whole
    path against the oracle's ES-kernel NUFFT; the oracle interpolates a sample of particles."""
    pos, c = gen.make_config_positions("cfg3", n_p=128)
    n = pos.shape[0]
    m, box = c["m"], c["box"]
    ctx = pm.pm_create(nufft_params(pm, m, box, n))
    w, beta = ctx.nufft_width, ctx.nufft_beta
    f = torch.empty(n, 3, device="cuda")
    pm.pm_force(ctx, dev(pos), f)
    pm.pm_destroy(ctx)
    fine = no.es_spread(pos, 2 * m, box, w, beta)
    g = no.nufft_kspace(fine, m, box, n, w, beta)
    idx = np.sort(np.random.default_rng(4245).choice(n, size=50_000, replace=False))
    ref = np.stack([no.es_interp(g[a], pos[idx], box, w, beta) for a in range(3)], axis=1)
    check("force/sampled=50000", f.cpu().numpy()[idx], ref, 1e-5)
