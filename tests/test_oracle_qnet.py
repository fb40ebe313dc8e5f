"""Pins the oracle's Q-network forward (Deep Q-Learning over 12 actions).

* hand special cases (one-hot / identity weights) whose outputs are known without running anything;
* an independent float64 torch.nn.functional reference (different library, different accumulation order) within 1e-5;
* argmax: lowest index on ties;  epsilon-greedy thresholds.
"""
import numpy as np
import torch

from oracle import oracle as O
from paper_2606_25082_b200 import workloads as W


def _zero_net(A=12, H=256):
    return W.QNetWeights(np.zeros((64, H), np.float32), np.zeros(H, np.float32), np.zeros((H, H), np.float32),
                         np.zeros(H, np.float32), np.zeros((H, A), np.float32), np.zeros(A, np.float32))


def test_bias_only_network():
    q = _zero_net()
    q.b3[:] = np.arange(12, dtype=np.float32) - 3.0
    x = np.random.default_rng(0).normal(size=(5, 64)).astype(np.float32)
    out, am = O.q_eval(q, x)
    assert np.array_equal(out, np.tile(q.b3, (5, 1))) and np.all(am == 11)


def test_one_hot_path_by_hand():
    # x[3] -> hidden1[7] (w=2, b=+1) -> relu -> hidden2[9] (w=-0.5, b=+4) -> relu -> q[5] (w=3, b=-1)
    q = _zero_net()
    q.W1[3, 7] = 2.0; q.b1[7] = 1.0
    q.W2[7, 9] = -0.5; q.b2[9] = 4.0
    q.W3[9, 5] = 3.0; q.b3[5] = -1.0
    x = np.zeros((3, 64), np.float32)
    x[0, 3] = 1.5      # h1 = 4   -> h2 = 2    -> q5 = 5
    x[1, 3] = -2.0     # h1 = relu(-3) = 0 -> h2 = 4 -> q5 = 11
    x[2, 3] = 10.0     # h1 = 21  -> h2 = relu(-6.5) = 0 -> q5 = -1
    out, am = O.q_eval(q, x)
    assert out[0, 5] == 5.0 and out[1, 5] == 11.0 and out[2, 5] == -1.0
    assert np.count_nonzero(out[:, np.arange(12) != 5]) == 0
    assert list(am) == [5, 5, 0]        # third row: q5 = -1 < 0 = all others -> lowest index among the zeros


def test_layout_is_in_by_out_row_major():
    # W[k][n]: a weight at (k=1, n=2) must connect input 1 to output 2, not the transpose
    q = _zero_net()
    q.W1[1, 2] = 1.0
    q.W2[2, 3] = 1.0
    q.W3[3, 4] = 1.0
    x = np.zeros((1, 64), np.float32); x[0, 1] = 7.0
    out, am = O.q_eval(q, x)
    assert out[0, 4] == 7.0 and am[0] == 4
    x = np.zeros((1, 64), np.float32); x[0, 2] = 7.0
    out, _ = O.q_eval(q, x)
    assert not out.any()


def test_against_float64_torch_reference():
    q = W.make_qnet(5, 12)
    rng = np.random.default_rng(1)
    x = rng.uniform(0, 4, size=(64, 64)).astype(np.float32)
    out, am = O.q_eval(q, x)
    t = lambda a: torch.from_numpy(np.asarray(a, dtype=np.float64))
    h1 = torch.relu(t(x) @ t(q.W1) + t(q.b1))
    h2 = torch.relu(h1 @ t(q.W2) + t(q.b2))
    ref = (h2 @ t(q.W3) + t(q.b3)).numpy()
    assert np.max(np.abs(out - ref) / np.maximum(1e-3, np.abs(ref))) < 1e-4
    assert np.max(np.abs(out - ref)) < 1e-5
    assert np.allclose(O.q_eval_f64(q, x), ref, rtol=1e-12, atol=1e-12)
    gap = np.sort(ref, axis=1)
    clear = (gap[:, -1] - gap[:, -2]) > 1e-4
    assert np.array_equal(am[clear], ref.argmax(axis=1)[clear])


def test_argmax_lowest_index_on_ties():
    q = _zero_net()
    q.b3[:] = [1, 5, 5, 2, 5, 0, 0, 0, 0, 0, 0, 0]
    _, am = O.q_eval(q, np.zeros((1, 64), np.float32))
    assert am[0] == 1


def test_epsilon_greedy_rates():
    # DQN policy in the oracle rollout: explore iff w_explore < round(eps 2^32); eps = 0 never explores, eps = 1 always
    wl = W.config_c4(2)
    r0 = O.rollout(wl.params, wl.seed, 0, algo=1, cfg0=0, policy=W.POLICY_DQN, qnet=wl.qnet, epsilon=0.0, want_states=True)
    _, am = O.q_eval(wl.qnet, r0.states[:24])
    assert np.array_equal(r0.actions, am)
    acts = []
    for e in range(40):
        r1 = O.rollout(wl.params, wl.seed, e, algo=1, cfg0=0, policy=W.POLICY_DQN, qnet=wl.qnet, epsilon=1.0)
        w = np.array([O.philox(k, 2, e, 0, wl.seed, 0) for k in range(24)], dtype=np.uint64)
        assert np.array_equal(r1.actions, ((w[:, 1] * 12) >> 32).astype(np.uint8))
        acts.append(r1.actions)
    acts = np.concatenate(acts)
    assert set(acts.tolist()) == set(range(12))
