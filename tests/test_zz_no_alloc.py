"""mig_q_forward_static -- the entry point that allocates nothing (its scratch is a file-scope static __device__ array of
libmigsim.so; include/migsim.h) -- against the existing tensor-core forward mig_dqn_q, on two calls in a row.

The second call uses a SMALLER network (hidden 128, 5 actions) and fewer rows than the first (hidden 256, 16 actions), so
that stale contents of the shared array -- action rows 5..15 of the split W3 copy, rows beyond n of the activations --
would show up if they were not cleared / ignored; a third call repeats the first one.  Tolerance: TOL = 1e-4 of max |Q|,
the bound the DQN tests use (tests/test_gpu_dqn.py); the two paths run the same kernels, so the results are in fact equal.

This file is named to be collected LAST (the suite runs with pytest -x) and passes alone in a fresh process as well as
after the other tests: it takes nothing from them and leaves no state but the array's contents."""
import numpy as np
import pytest
import torch

from paper_2606_25082_b200 import workloads as W

pytestmark = pytest.mark.gpu

TOL = 1e-4


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def both_paths(B, net, n, seed):
    """Q-values of `n` random states from the existing path (a mig_dqn handle, which allocates at create) and from the
    static entry point (device weights passed in, no handle)."""
    rng = np.random.default_rng(seed)
    s = dev(rng.normal(0, 1, (n, 64)).astype(np.float32))
    A = net.n_actions
    d = B.Dqn(net, 128, ((n + 127) // 128) * 128, 0.9, 0.01, 1)
    want = d.q(s).cpu().numpy()
    d.close()
    w = [dev(np.asarray(x, np.float32)) for x in (net.W1, net.b1, net.W2, net.b2, net.W3, net.b3)]
    q = torch.full((n, A), float("nan"), dtype=torch.float32, device="cuda")
    B.q_forward_static(*w, s, q)
    torch.cuda.synchronize()
    return q.cpu().numpy(), want


def test_static_forward_matches_the_allocating_path_on_calls_in_a_row():
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2606_25082_b200 import binding as B
    big = W.make_qnet(5, n_actions=16, hidden=256)
    small = W.make_qnet(6, n_actions=5, hidden=128)
    for k, (net, n) in enumerate([(big, B.Q_STATIC_MAX_ROWS), (small, 1000), (big, 77), (small, 129)]):
        got, want = both_paths(B, net, n, 100 + k)
        assert got.shape == want.shape and np.isfinite(got).all(), k
        err = np.abs(got - want).max()
        assert err <= TOL * np.abs(want).max(), (k, err, np.abs(want).max())


def test_static_forward_is_the_double_precision_forward_too():
    # not only equal to the other CUDA path: within the same tolerance of the oracle's double-precision network
    from oracle import oracle as O
    from paper_2606_25082_b200 import binding as B
    net = W.make_qnet(9, n_actions=12, hidden=256)
    rng = np.random.default_rng(9)
    s = rng.normal(0, 1, (300, 64)).astype(np.float32)
    w = [dev(np.asarray(x, np.float32)) for x in (net.W1, net.b1, net.W2, net.b2, net.W3, net.b3)]
    q = torch.empty((300, 12), dtype=torch.float32, device="cuda")
    for _ in range(2):                                           # two calls in a row on the same array
        q.fill_(float("nan"))
        B.q_forward_static(*w, dev(s), q)
        torch.cuda.synchronize()
        want = O.Dqn(net, 0.9, 0.01).q(s)
        assert np.abs(q.cpu().numpy() - want).max() <= TOL * np.abs(want).max()


def test_static_forward_rejects_what_does_not_fit():
    from paper_2606_25082_b200 import binding as B
    net = W.make_qnet(5, n_actions=12, hidden=256)
    w = [dev(np.asarray(x, np.float32)) for x in (net.W1, net.b1, net.W2, net.b2, net.W3, net.b3)]
    n = B.Q_STATIC_MAX_ROWS + 1
    s = torch.zeros((n, 64), dtype=torch.float32, device="cuda")
    q = torch.zeros((n, 12), dtype=torch.float32, device="cuda")
    with pytest.raises(B.MigError) as ei:
        B.q_forward_static(*w, s, q)
    assert ei.value.code == B.MIG_EINVAL and "MIG_Q_STATIC_MAX_ROWS" in str(ei.value)
    bad = W.make_qnet(5, n_actions=12, hidden=64)                # hidden must be 128 or 256
    wb = [dev(np.asarray(x, np.float32)) for x in (bad.W1, bad.b1, bad.W2, bad.b2, bad.W3, bad.b3)]
    with pytest.raises(B.MigError) as ei:
        B.q_forward_static(*wb, s[:8], q[:8])
    assert ei.value.code == B.MIG_EINVAL
