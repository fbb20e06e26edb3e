"""pm_mesh_power_noalloc (the allocation-free shell binning, scratch in a static __device__ array) against the
existing path, pm_power_spectrum, on two calls in a row.  Collected last on purpose (file name): the suite runs with
pytest -x, so a failure here hides nothing behind it.

The existing path bins the spectrum of the density it assigns itself; the new entry point bins spectra the caller
holds.  The test therefore rebuilds that spectrum with public calls (pm_assign of the same particles, torch's R2C
transform) and compares the three outputs bin by bin, at the tolerance of test_power_spectrum_parity."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

from pm_inputs import generators as gen

from parity_util import check

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def pm():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2510_05206_b200 as pm_

    return pm_


def dev(x):
    return torch.from_numpy(np.ascontiguousarray(x)).cuda()


def spectrum_of(pm, ctx, pos_dev, m):
    mesh = torch.zeros(m, m, m, device="cuda")
    pm.pm_assign(ctx, pos_dev, None, mesh)
    return torch.view_as_real(torch.fft.rfftn(mesh)).contiguous()


def test_noalloc_matches_power_spectrum_twice_in_a_row(pm):
    """Two calls back to back with different particle sets and bin counts: the second call finds the first call's
    sums in the shared scratch array and must clear them.  The third call is a cross spectrum."""
    pos, c = gen.make_config_positions("cfg1", n_p=64)
    n, m, box = pos.shape[0], c["m"], c["box"]
    pos2 = pos.copy()
    pos2[:, 0] = np.mod(pos2[:, 0] + np.float32(3.0 * box / m), np.float32(box))
    pos3 = gen.uniform_random(n // 2, box, 77)
    ctx = pm.pm_create(pm.PMParams(m=m, box=box, max_particles=n, worder=2, interlace=0))
    sets = {"a": dev(pos), "b": dev(pos2), "c": dev(pos3)}
    spec = {k: spectrum_of(pm, ctx, v, m) for k, v in sets.items()}
    cases = [("first", "a", None, 40), ("second", "c", None, 24), ("cross", "a", "b", 40)]
    # every input and output exists before the calls under test; the calls run back to back
    outs = {name: [torch.full((nb,), -1.0, dtype=torch.float64, device="cuda") for _ in range(3)]
            for name, _, _, nb in cases}
    for name, ka, kb, nb in cases:
        na, nb_ = sets[ka].shape[0], sets[kb or ka].shape[0]
        pm.pm_mesh_power_noalloc(spec[ka], m, box, box ** 3 / (float(na) * float(nb_)), *outs[name],
                                 spec_b=spec[kb] if kb else None)
    torch.cuda.synchronize()
    for name, ka, kb, nb in cases:
        k, P, cnt = (torch.zeros(nb, dtype=torch.float64, device="cuda") for _ in range(3))
        pm.pm_power_spectrum(ctx, sets[ka], k, P, cnt, pos2=sets[kb] if kb else None, deconvolve=False)
        k0, P0, c0 = (t.cpu().numpy() for t in outs[name])
        assert np.array_equal(c0, cnt.cpu().numpy()), name  # mode counts: integer work, exact
        assert np.abs(k0 - k.cpu().numpy()).max() <= 1e-12 * k.max().item(), name
        check(f"{name}/P", P0, P.cpu().numpy(), 2e-5 if kb else 1e-5, maxabs_tol=1e-3)
    pm.pm_destroy(ctx)


def test_noalloc_rejects_sizes_beyond_the_static_array(pm):
    m = 16
    spec = torch.zeros(m, m, m // 2 + 1, 2, device="cuda")
    nb = pm.NOALLOC_MAX_BINS + 1
    k, P, cnt = (torch.zeros(nb, dtype=torch.float64, device="cuda") for _ in range(3))
    with pytest.raises(pm.PMError, match="PM_NOALLOC_MAX_BINS"):
        pm.pm_mesh_power_noalloc(spec, m, 1.0, 1.0, k, P, cnt)
    # the largest size it accepts still runs (all but the lowest bins are empty on a 16^3 mesh)
    k, P, cnt = (torch.full((pm.NOALLOC_MAX_BINS,), -1.0, dtype=torch.float64, device="cuda") for _ in range(3))
    pm.pm_mesh_power_noalloc(spec, m, 1.0, 1.0, k, P, cnt)
    torch.cuda.synchronize()
    assert float(cnt.sum()) > 0 and float(P.abs().max()) == 0.0 and float(cnt[20:].sum()) == 0.0
