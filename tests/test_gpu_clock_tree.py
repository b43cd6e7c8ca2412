"""The expiry tournament tree of the cumulative clock (Theorem 2; kc.h) against the
oracle's flat rule F = {i : c_i <= 4 (S - S_i)}: the same set, step after step, with certificates that
sit exactly on the boundary, zero and infinite clearances, and sizes that are not multiples of the
fanout."""
import numpy as np
import pytest
import torch

import oracle
from paper_2606_18314_b200 import binding as kc
from _util import dev

pytestmark = pytest.mark.gpu


def _ids(F, nF):
    torch.cuda.synchronize()
    return np.sort(F.cpu().numpy()[: int(nF.item())])


@pytest.mark.parametrize("N", [1, 31, 32, 33, 1023, 1025, 40000, 1048577])
def test_tree_gives_the_flat_rule_step_after_step(N):
    rng = np.random.default_rng(N)
    c = (rng.random(N) ** 2 * 0.02).astype(np.float32)
    c[rng.random(N) < 0.01] = 0.0                                   # duplicates: always expired
    c[rng.random(N) < 0.01] = np.inf                                # (a lone point: never)
    stamp = np.zeros(N, np.float32)
    S = 0.0
    C, ST = dev(c), dev(stamp)
    tree = kc.kc_clock_tree_build(C, ST)
    assert tree.numel() == (N + 31) // 32 + ((N + 31) // 32 + 31) // 32
    S_dev = [torch.zeros(1, dtype=torch.float64, device="cuda"), torch.zeros(1, dtype=torch.float64, device="cuda")]
    sizes = []
    for step in range(12):
        eps = np.float32([1e-6, 1e-6, 1e-5, 2e-4, 1e-3, 1e-3, 1e-5, 1e-6, 2e-4, 1e-3, 1e-6, 1e-5][step])
        if step == 5:
            # certificates exactly on the boundary: c = 4 (S_next - stamp) in float64 terms
            S_next = np.float64(S) + np.float64(eps)
            k = rng.choice(N, max(1, N // 50), replace=False)
            c[k] = (4.0 * (S_next - stamp[k].astype(np.float64))).astype(np.float32)
            C = dev(c)
            kc.kc_clock_tree_build(C, ST, tree)
        S, flags, want = oracle.clock_frontier(c, stamp, S, eps)
        F, nF = kc.kc_frontier_classify_clock_tree(C, ST, tree, S_dev[0], dev(np.array([eps], np.float32)), S_dev[1])
        S_dev.reverse()
        assert float(S_dev[0].item()) == S
        got = _ids(F, nF)
        assert np.array_equal(got, want), f"N={N} step {step}: {got.size} vs {want.size}"
        sizes.append(want.size)
        # "recompute" the expired certificates: new clearances, stamped with the clock
        c[want] = (rng.random(want.size) ** 2 * 0.02).astype(np.float32)
        stamp[want] = oracle.clock_stamp(S)
        C, ST = dev(c), dev(stamp)
        kc.kc_clock_tree_update(tree, C, ST, F, nF)
        full = kc.kc_clock_tree_build(C, ST)
        torch.cuda.synchronize()
        assert torch.equal(tree, full), f"N={N} step {step}: updated tree differs from a rebuilt one"
    assert N < 1000 or (min(sizes) < N // 16 and max(sizes) > 0)      # both update shapes were used


def test_tree_argument_errors():
    c = torch.zeros(64, device="cuda")
    tree = kc.kc_clock_tree_build(c, c.clone())
    S = torch.zeros(1, dtype=torch.float64, device="cuda")
    with pytest.raises(kc.KcError):
        kc.kc_frontier_classify_clock_tree(c, c, tree, S, torch.zeros(1, device="cuda"), S)
    assert kc.lib().kc_clock_tree_floats(0) == 0 and kc.lib().kc_clock_tree_floats(1025) == 33 + 2
