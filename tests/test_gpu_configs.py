"""GPU parity at the BASELINE.json configurations, in the launch configuration bench.py times.

cfg2 (K=24, D=500, honest blocking) is small enough for a full element-by-element comparison.  cfg3-cfg5 are
compared on sampled sigma blocks the oracle can compute one by one (oracle.opair_sigma(only_out=...)): the
largest block, the smallest block and a seeded random handful, plus properties that hold at any size
(Hermiticity, bitwise reproducibility, theta == Rayleigh quotient of the returned Ritz vector).
Bar: max|d sigma| / ||sigma||_2 <= 1e-11 (BASELINE.json north_star).
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

import oracle  # noqa: E402
from dmrg_workload.problem import make_config, random_psi  # noqa: E402

TOL_SIGMA = 1e-11


def _gpu():
    import paper_2311_02854_b200 as g
    if not torch.cuda.is_available():
        pytest.fail("gpu-marked test needs a CUDA device")
    return g


def _sigma(plan, v):
    d = torch.from_numpy(v).cuda()
    o = torch.empty_like(d)
    plan.sigma(d, o, torch.cuda.current_stream())
    torch.cuda.synchronize()
    return o.cpu().numpy()


def _sample_blocks(pr, plan, budget_flops, seed=0):
    """Seeded random sigma blocks whose estimated oracle cost (share of psi x total flops) fits the budget,
    always including the smallest block and the largest block that fits."""
    lay = np.asarray(pr.layout)
    size = (lay[:, 4] * lay[:, 5]).astype(float)
    cost = size / size.sum() * plan.stats()["canon_flops"]
    rng = np.random.default_rng(seed)
    pick, acc = [int(np.argmin(size))], 0.0
    fits = np.nonzero(cost <= 0.5 * budget_flops)[0]
    if len(fits):
        big = int(fits[np.argmax(size[fits])])
        pick.append(big)
        acc += cost[big]
    for b in rng.permutation(len(lay)):
        if acc + cost[b] > budget_flops:
            continue
        pick.append(int(b))
        acc += cost[b]
        if len(pick) >= 10:
            break
    return sorted(set(pick))


def _block_err(pr, got, ref, blocks):
    lay = np.asarray(pr.layout)
    err = 0.0
    for b in blocks:
        o, cnt = int(lay[b][6]), int(lay[b][4] * lay[b][5])
        err = max(err, float(np.abs(got[o:o + cnt] - ref[o:o + cnt]).max()))
    return err


def test_cfg2_full_parity_and_davidson():
    g = _gpu()
    pr = make_config("cfg2")
    ops, plan = g.load_problem(pr)
    assert np.array_equal(plan.psi_layout(), pr.layout)
    psi = random_psi(pr.psi_size, 5)
    ref = oracle.opair_sigma(pr, psi)
    got = _sigma(plan, psi)
    assert np.abs(got - ref).max() / np.linalg.norm(ref) <= TOL_SIGMA
    assert np.array_equal(got, _sigma(plan, psi))                     # bitwise reproducible
    hd = torch.empty(pr.psi_size, dtype=torch.float64, device="cuda")
    plan.hdiag(hd, torch.cuda.current_stream())
    torch.cuda.synchronize()
    ref_hd = oracle.opair_hdiag(pr)
    assert np.abs(hd.cpu().numpy() - ref_hd).max() <= 1e-12 * max(1.0, np.abs(ref_hd).max())
    # the configured run: 20 Davidson iterations from the random psi
    x = torch.from_numpy(psi).cuda()
    res = plan.davidson(x, max_iter=20, max_space=20, tol=0.0, stream=torch.cuda.current_stream())
    assert res["iters"] == 20
    xn = x.cpu().numpy()
    hx = oracle.opair_sigma(pr, xn)                                   # one oracle H psi on the GPU's Ritz vector
    assert abs(xn @ hx - res["energy"]) <= 1e-9
    assert abs(np.linalg.norm(hx - res["energy"] * xn) - res["resid"]) <= 1e-8
    assert np.all(np.diff(res["thetas"]) <= 1e-12)                    # Ritz values decrease monotonically
    plan.destroy()
    ops.free()


@pytest.mark.parametrize("name,budget", [("cfg3", 2.5e11), ("cfg4", 2.5e11), ("cfg5", 4e11)])
def test_direct_configs_sampled_parity(name, budget):
    g = _gpu()
    pr = make_config(name)
    ops, plan = g.load_problem(pr)
    assert np.array_equal(plan.psi_layout(), pr.layout)
    psi, phi = random_psi(pr.psi_size, 5), random_psi(pr.psi_size, 6)
    s_psi = _sigma(plan, psi)
    assert np.array_equal(s_psi, _sigma(plan, psi))                   # bitwise reproducible
    s_phi = _sigma(plan, phi)
    nrm = np.linalg.norm(s_psi)
    assert abs(phi @ s_psi - s_phi @ psi) <= 1e-11 * nrm               # Hermiticity (pin 3) at full size
    # a short Davidson; then ONE oracle call checks sampled blocks of H psi and of H x (x = Ritz vector)
    x = torch.from_numpy(psi).cuda()
    res = plan.davidson(x, max_iter=4, max_space=4, tol=0.0, stream=torch.cuda.current_stream())
    xn = x.cpu().numpy()
    hx = _sigma(plan, xn)
    assert abs(xn @ hx - res["energy"]) <= 1e-9 * max(1.0, abs(res["energy"]))      # theta is the Rayleigh quotient
    assert abs(np.linalg.norm(hx - res["energy"] * xn) - res["resid"]) <= 1e-8 * max(1.0, res["resid"])
    blocks = _sample_blocks(pr, plan, budget)
    ref, st = oracle.opair_sigma(pr, psi, only_out=blocks, return_stats=True)
    assert st["tasks"] > 0
    assert _block_err(pr, s_psi, ref, blocks) / nrm <= TOL_SIGMA
    lay = np.asarray(pr.layout)
    small = [int(np.argmin(lay[:, 4] * lay[:, 5]))]                    # the smallest block: cheap second oracle call
    ref_x = oracle.opair_sigma(pr, xn, only_out=small)
    assert _block_err(pr, hx, ref_x, small) / np.linalg.norm(hx) <= TOL_SIGMA
    s = plan.stats()
    assert s["canon_flops"] > 0 and s["padded_flops"] >= s["s1_flops"] + s["s2_flops"] - 1
    plan.destroy()
    ops.free()
