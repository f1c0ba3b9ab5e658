"""gdn_compute_gates_static (include/gdn.h): the gates of PAPER.md Eq. 13-15 through the entry point that allocates
nothing (its scratch is a file-scope static __device__ array of the library).  Collected last on purpose (the suite
runs with pytest -x): checked against the existing path, gdn_compute_gates, on two calls in a row that share the array,
and against the oracle; sizes beyond the static scratch are refused.  Runs alone in a fresh process or after the other
tests alike (it needs no plan for the new entry point and leaves nothing behind)."""
import numpy as np
import pytest
import torch

import paper_2605_30409_b200 as gdn
from paper_2605_30409_b200 import inputs as gin

pytestmark = pytest.mark.gpu
DEV = "cuda:0"
RTOL, ATOL = 2e-5, 2e-6          # the tolerance of tests/test_gpu_frontend.py::test_gates_match_oracle_and_are_deterministic

# (B, H, G, F, D): the paper's production chunk, then a different shape with fewer splits, strides and frames, so that
# the second call finds the first call's partial sums and counters in the shared array
CALLS = [(1, 20, 880, 3, 112), (2, 3, 100, 4, 128)]


def _existing_path(fi, B, H, T, D, G, log_alpha, dev):
    flags = gdn.GDN_FLAG_NORMALIZER | (gdn.GDN_FLAG_LOG_ALPHA if log_alpha else 0)
    a = torch.full((B, H, T // G), float("nan"), device=DEV)
    b = torch.full((B, H, T), float("nan"), device=DEV)
    with gdn.GdnPlan(B=B, H=H, T=T, d_k=D, d_v=D, group=G, flags=flags) as p:
        ga = gdn.make_gate_args(dev["x"], dev["w_alpha"], dev["b_alpha"], dev["a_log"], dev["w_beta"], dev["b_beta"])
        p.compute_gates(ga, a, b)
        torch.cuda.synchronize()
    return a.cpu(), b.cpu()


@pytest.mark.parametrize("log_alpha", [False, True])
def test_static_scratch_gates_match_the_existing_path_on_two_calls_in_a_row(log_alpha):
    from oracle import frontend as fe
    results = []
    for i, (B, H, G, F, D) in enumerate(CALLS):           # the two calls of the new entry point, back to back
        T = G * F
        wl = gin.GdnWorkload("static_gates", B, H, T, D, D, group=G, seed=900 + i)
        fi = gin.make_frontend_inputs(wl)
        dev = {n: fi[n].to(DEV) for n in ("x", "w_alpha", "b_alpha", "a_log", "w_beta", "b_beta")}
        a = torch.full((B, H, F), float("nan"), device=DEV)
        b = torch.full((B, H, T), float("nan"), device=DEV)
        ga = gdn.make_gate_args(dev["x"], dev["w_alpha"], dev["b_alpha"], dev["a_log"], dev["w_beta"], dev["b_beta"])
        gdn.gdn_compute_gates_static(ga, B, T, H, D, G, log_alpha, a, b)
        results.append((fi, dev, a, b))
    torch.cuda.synchronize()
    for (B, H, G, F, D), (fi, dev, a, b) in zip(CALLS, results):
        T = G * F
        want_a, want_b = _existing_path(fi, B, H, T, D, G, log_alpha, dev)
        np.testing.assert_allclose(a.cpu().numpy(), want_a.numpy(), rtol=RTOL, atol=ATOL)
        np.testing.assert_allclose(b.cpu().numpy(), want_b.numpy(), rtol=RTOL, atol=ATOL)
        alpha, la, beta = fe.gates(fi["x"], fi["w_alpha"], fi["b_alpha"], fi["a_log"], fi["w_beta"], fi["b_beta"], group=G)
        np.testing.assert_allclose(a.cpu().double().numpy(), la if log_alpha else alpha, rtol=RTOL, atol=ATOL)
        np.testing.assert_allclose(b.cpu().double().numpy(), beta, rtol=RTOL, atol=ATOL)


def test_static_scratch_gates_refuse_sizes_beyond_the_array():
    B, H, G, F, D = 1, 4100, 8, 1, 64                      # 4100 frame-heads > 4096
    T = G * F
    x = torch.zeros(B, T, H, D, device=DEV, dtype=torch.bfloat16)
    w = torch.zeros(H, D, device=DEV)
    v = torch.zeros(H, device=DEV)
    a = torch.full((B, H, F), 7.0, device=DEV)
    b = torch.full((B, H, T), 7.0, device=DEV)
    ga = gdn.make_gate_args(x, w, v, v, w, v)
    with pytest.raises(gdn.GdnError) as ei:
        gdn.gdn_compute_gates_static(ga, B, T, H, D, G, False, a, b)
    assert ei.value.status == gdn.GDN_ERR_UNSUPPORTED and "4096" in str(ei.value)
    torch.cuda.synchronize()
    assert (a == 7.0).all() and (b == 7.0).all()           # nothing was launched
    with pytest.raises(gdn.GdnError) as ei:                # a head dim the kernel has no lanes for
        gdn.gdn_compute_gates_static(ga, 1, 8, 4, 136, 8, False, a, b)
    assert ei.value.status == gdn.GDN_ERR_UNSUPPORTED
