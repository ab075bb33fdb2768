"""dmrg_dots_static (include/dmrg_sigma.h): the Davidson dot-product kernels on a file-scope device scratch array,
for callers that may not allocate.  Checked against the existing path -- the same kernels on dmrg_davidson's
cudaMalloc'ed workspace, read back through the solver's outputs -- on two calls in a row, and against plain FP64 sums.

Collected last on purpose (file name): a failure here must not hide the parity tests under `pytest -x`.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from dmrg_workload.problem import make_blocked_problem, random_psi  # noqa: E402

RTOL = 1e-11   # the sigma tolerance of the parity tests (tests/test_gpu_parity.py: TOL_SIGMA)


def _gpu():
    import paper_2311_02854_b200 as g
    if not torch.cuda.is_available():
        pytest.fail("gpu-marked test needs a CUDA device")
    return g


def test_dots_static_matches_the_davidson_path_twice():
    g = _gpu()
    pr = make_blocked_problem(K=10, nL=4, N_tot=10, D=60, seed=3)
    ops, plan = g.load_problem(pr)
    st = torch.cuda.current_stream()
    n = pr.psi_size
    x0 = torch.from_numpy(random_psi(n, 21)).cuda()
    x0 /= x0.norm()
    # existing path: one Davidson iteration = theta = b0 . (H b0) and |r| = sqrt(r . r), r = H b0 - theta b0, both
    # formed by dots_partial_kernel / dots_final_kernel on the workspace ws_ensure cudaMalloc's
    x = x0.clone()
    res = plan.davidson(x, max_iter=1, max_space=2, tol=1e-30, stream=st)
    # new path: the same quantities through the static-scratch entry point; b0 and w0 stacked as two vectors
    bw = torch.empty(2, n + (n & 1), dtype=torch.float64, device="cuda")[:, :n]
    bw[0] = x0
    plan.sigma(bw[0], bw[1], st)
    out = torch.full((g.DOTS_STATIC_MAX_VECTORS,), float("nan"), dtype=torch.float64, device="cuda")
    for call in range(2):   # two calls in a row: the second one finds the first one's partial sums in the scratch
        out.fill_(float("nan"))
        g.dots_static(bw, bw[1], out, st)            # call A: [b0 . w0, w0 . w0]
        theta, ww = out[:2].tolist()
        r = bw[1] - theta * bw[0]
        g.dots_static(r, r, out[2:], st)             # call B: one vector, other data, same scratch
        rn = float(out[2].sqrt())
        assert abs(theta - res["energy"]) <= RTOL * max(1.0, abs(res["energy"])), (call, theta, res["energy"])
        assert abs(rn - res["resid"]) <= RTOL * max(1.0, res["resid"]), (call, rn, res["resid"])
        assert abs(ww - float(bw[1].double() @ bw[1])) <= RTOL * ww, call
        assert torch.isnan(out[3:]).all()            # nothing written beyond m outputs
    # a full block of vectors with a ragged length, after the small calls (stale partial sums of rows 0-1 in place)
    m, nn = g.DOTS_STATIC_MAX_VECTORS, 100003
    gen = torch.Generator(device="cuda").manual_seed(5)
    V = torch.randn(m, nn + 1, dtype=torch.float64, device="cuda", generator=gen)[:, :nn]
    w = torch.randn(nn, dtype=torch.float64, device="cuda", generator=gen)
    ref = (V.cpu().numpy() * w.cpu().numpy()).sum(axis=1)
    scale = np.abs(V.cpu().numpy() * w.cpu().numpy()).sum(axis=1)
    first = None
    for call in range(2):
        g.dots_static(V, w, out, st)
        got = out.cpu().numpy()
        assert np.all(np.abs(got - ref) <= RTOL * scale), call
        first = got if first is None else first
        assert np.array_equal(got, first)            # fixed summation tree: bitwise the same on the second call
    # n = 0: zeros, not stale sums
    assert g.lib().dmrg_dots_static(V.data_ptr(), V.stride(0), m, w.data_ptr(), 0, out.data_ptr(), st.cuda_stream) == 0
    assert torch.equal(out, torch.zeros_like(out))
    plan.destroy()
    ops.free()


def test_dots_static_rejects_sizes_beyond_the_scratch():
    g = _gpu()
    m = g.DOTS_STATIC_MAX_VECTORS + 1
    V = torch.zeros(m, 8, dtype=torch.float64, device="cuda")
    out = torch.zeros(m, dtype=torch.float64, device="cuda")
    with pytest.raises(g.DmrgError) as ei:
        g.dots_static(V, V[0], out)
    assert ei.value.code == -1 and str(g.DOTS_STATIC_MAX_VECTORS) in str(ei.value)
