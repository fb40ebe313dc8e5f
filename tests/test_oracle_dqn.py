"""Pins for the DQN training oracle (oracle/dqn_oracle.c; readings #33-#36), written before
the CUDA training path: a hand-worked one-neuron update, a finite-difference check of every gradient entry, the special
cases (lr = 0, done, gamma = 0, dead ReLU, frozen target), agreement of its forward with the already pinned double-precision
Q evaluation, and the replay sampler against an independent computation from the pinned Philox.

Mutations of dqn_oracle.c these were checked to kill: delta / 2B (gradient halved); relu' taken on z2 of the TARGET pass;
max replaced by Q_target(s', a); (1 - done) dropped; W2 transposed in the backward pass; gb1 from dz2; target updated by
the step; sampler reading word 1; index = w % size.
"""
import numpy as np
import pytest

from oracle import oracle as O
from paper_2606_25082_b200 import workloads as W


def small_net(seed, H=8, A=3):
    rng = np.random.default_rng(seed)
    return W.QNetWeights(W1=rng.normal(0, 0.3, (64, H)).astype(np.float32), b1=rng.normal(0, 0.1, H).astype(np.float32),
                         W2=rng.normal(0, 0.4, (H, H)).astype(np.float32), b2=rng.normal(0, 0.1, H).astype(np.float32),
                         W3=rng.normal(0, 0.5, (H, A)).astype(np.float32), b3=rng.normal(0, 0.1, A).astype(np.float32))


def batch(seed, B, A=3):
    rng = np.random.default_rng(seed)
    s = rng.normal(0, 1, (B, 64)).astype(np.float32)
    s2 = rng.normal(0, 1, (B, 64)).astype(np.float32)
    a = rng.integers(0, A, B).astype(np.uint8)
    r = rng.normal(0, 1, B).astype(np.float32)
    done = (rng.random(B) < 0.3).astype(np.uint8)
    return s, a, r, s2, done


def test_one_neuron_update_by_hand():
    # H = 1, A = 1: W1[0][0] = 2, W2 = 3, W3 = 0.5, all biases 0.  s = e_0: h1 = 2, h2 = 6, Q = 3.  s' = e_0 / 2: Q' = 1.5.
    # r = 1, gamma = 0.9: y = 2.35, delta = 0.65, L = 0.65^2 / 2 = 0.21125.  dQ = 0.65: gb3 = 0.65, gW3 = 6 * 0.65 = 3.9,
    # dz2 = 0.65 * 0.5 = 0.325 = gb2, gW2 = 2 * 0.325 = 0.65, dz1 = 0.325 * 3 = 0.975 = gb1 = gW1[0][0].
    # lr = 0.1: W1[0][0] = 1.9025, b1 = -0.0975, W2 = 2.935, b2 = -0.0325, W3 = 0.11, b3 = -0.065.
    W1 = np.zeros((64, 1), np.float32); W1[0, 0] = 2.0
    net = W.QNetWeights(W1=W1, b1=np.zeros(1, np.float32), W2=np.full((1, 1), 3.0, np.float32), b2=np.zeros(1, np.float32),
                        W3=np.full((1, 1), 0.5, np.float32), b3=np.zeros(1, np.float32))
    d = O.Dqn(net, gamma=0.9, lr=0.1)
    s = np.zeros((1, 64), np.float32); s[0, 0] = 1.0
    s2 = np.zeros((1, 64), np.float32); s2[0, 0] = 0.5
    assert abs(d.q(s)[0, 0] - 3.0) < 1e-15 and abs(d.q(s2, which=1)[0, 0] - 1.5) < 1e-15
    loss, g = d.loss_grad(s, [0], [1.0], s2, [0])
    gW1, gb1, gW2, gb2, gW3, gb3 = d.split(g)
    y = 1.0 + float(np.float64(0.9) * 1.5)
    delta = 3.0 - y
    assert abs(loss - delta * delta / 2) < 1e-15 and abs(loss - 0.21125) < 1e-12
    assert abs(gb3[0] - 0.65) < 1e-12 and abs(gW3[0, 0] - 3.9) < 1e-12 and abs(gb2[0] - 0.325) < 1e-12
    assert abs(gW2[0, 0] - 0.65) < 1e-12 and abs(gb1[0] - 0.975) < 1e-12 and abs(gW1[0, 0] - 0.975) < 1e-12
    assert not gW1[1:].any()
    assert abs(d.train_step(s, [0], [1.0], s2, [0]) - 0.21125) < 1e-12
    W1n, b1n, W2n, b2n, W3n, b3n = d.split(d.params())
    for got, want in ((W1n[0, 0], 1.9025), (b1n[0], -0.0975), (W2n[0, 0], 2.935), (b2n[0], -0.0325), (W3n[0, 0], 0.11), (b3n[0], -0.065)):
        assert abs(got - want) < 1e-12, (got, want)
    assert np.array_equal(d.params(1), np.concatenate([W1.ravel(), [0], [3.0], [0], [0.5], [0]]))     # the target is frozen


def test_gradient_against_finite_differences():
    net = small_net(1)
    d = O.Dqn(net, gamma=0.95, lr=0.0)
    d.set_params(d.params() + np.random.default_rng(9).normal(0, 0.05, d.n), which=1)     # a target that differs from the online net
    s, a, r, s2, done = batch(2, 7)
    loss, g = d.loss_grad(s, a, r, s2, done)
    theta = d.params()
    eps = 1e-6
    worst = 0.0
    for i in range(d.n):                                      # every parameter: 64*8 + 8 + 64 + 8 + 24 + 3 = 619
        for sign, store in ((+1, "p"), (-1, "m")):
            t = theta.copy(); t[i] += sign * eps
            d.set_params(t)
            if sign > 0:
                lp, _ = d.loss_grad(s, a, r, s2, done, want_grad=False)
            else:
                lm, _ = d.loss_grad(s, a, r, s2, done, want_grad=False)
        fd = (lp - lm) / (2 * eps)
        worst = max(worst, abs(fd - g[i]) / max(1e-3, abs(g[i])))
    assert worst < 1e-5, worst
    d.set_params(theta)
    assert np.abs(g).max() > 1e-3 and loss > 0


def test_special_cases():
    net = small_net(3)
    s, a, r, s2, done = batch(4, 9)
    d = O.Dqn(net, gamma=0.9, lr=0.0)
    before = d.params()
    d.train_step(s, a, r, s2, done)
    assert np.array_equal(d.params(), before) and np.array_equal(d.params(1), before)      # lr = 0: identity
    # done = 1 everywhere or gamma = 0: the target is the reward alone, s' does not matter
    l1, g1 = O.Dqn(net, 0.9, 0.1).loss_grad(s, a, r, s2, np.ones(9, np.uint8))
    l2, g2 = O.Dqn(net, 0.0, 0.1).loss_grad(s, a, r, s2 * 3 + 1, None)
    assert l1 == l2 and np.array_equal(g1, g2)
    q = O.Dqn(net, 0.9, 0.1).q(s)
    assert abs(l1 - float(np.sum((q[np.arange(9), a] - r.astype(np.float64)) ** 2) / 18)) < 1e-12
    # the step leaves the target alone; sync copies the online network
    d = O.Dqn(net, 0.9, 0.05)
    t0 = d.params(1)
    for _ in range(3):
        d.train_step(s, a, r, s2, done)
    assert np.array_equal(d.params(1), t0) and not np.array_equal(d.params(0), t0)
    d.sync_target()
    assert np.array_equal(d.params(1), d.params(0))
    # a dead ReLU passes no gradient: very negative b1 kills the first layer -> gW1, gb1, gW2 are zero, gb2 is not
    dead = small_net(3); dead.b1[:] = -1e3
    _, g = O.Dqn(dead, 0.9, 0.1).loss_grad(s, a, r, s2, done)
    dd = O.Dqn(dead, 0.9, 0.1)
    gW1, gb1, gW2, gb2, gW3, gb3 = dd.split(g)
    assert not gW1.any() and not gb1.any() and not gW2.any() and gb2.any() and gb3.any()
    # only the taken action's output column receives gradient
    _, g = O.Dqn(net, 0.9, 0.1).loss_grad(s[:1], a[:1], r[:1], s2[:1], done[:1])
    gW3 = O.Dqn(net, 0.9, 0.1).split(g)[4]
    assert gW3[:, int(a[0])].any() and not np.delete(gW3, int(a[0]), axis=1).any()


def test_forward_agrees_with_the_pinned_double_precision_network():
    net = W.make_qnet(5, n_actions=12, hidden=64)
    s = np.random.default_rng(6).normal(0, 1, (20, 64)).astype(np.float32)
    assert np.allclose(O.Dqn(net, 0.9, 0.1).q(s), O.q_eval_f64(net, s), rtol=1e-13, atol=1e-13)


def test_loss_is_the_squared_td_error_with_the_max_over_the_target_network():
    # the loss recomputed from the two (separately pinned) forward passes: y = r + gamma (1 - done) max_a' Q_target(s', a')
    net = W.make_qnet(11, n_actions=12, hidden=32)
    s, a, r, s2, done = batch(12, 50, A=12)
    d = O.Dqn(net, gamma=0.8, lr=0.1)
    d.set_params(d.params() + np.random.default_rng(13).normal(0, 0.1, d.n), which=1)
    q, qt = d.q(s), d.q(s2, which=1)
    y = r.astype(np.float64) + np.float64(0.8) * (1 - done) * qt.max(axis=1)
    want = float(np.sum((q[np.arange(50), a] - y) ** 2) / 100.0)
    loss, _ = d.loss_grad(s, a, r, s2, done)
    assert abs(loss - want) < 1e-12 * max(1.0, want)
    assert np.any(qt.argmax(axis=1) != a)                      # (so that max != Q_target(s', a))


def test_loss_goes_down_on_a_fixed_batch():
    net = small_net(7)
    s, a, r, s2, done = batch(8, 64)
    d = O.Dqn(net, gamma=0.9, lr=0.05)
    losses = [d.train_step(s, a, r, s2, done) for _ in range(30)]
    assert losses[-1] < 0.7 * losses[0] and all(l2 < l1 * 1.001 for l1, l2 in zip(losses, losses[1:]))


def test_replay_sampler_is_philox_stream_3():
    seed, step, size, B = 0x1234567855AA, 17, 1000, 4096
    idx = O.replay_sample(seed, step, size, B)
    want = np.array([(int(O.philox(b, 3, step, 0, seed & 0xFFFFFFFF, seed >> 32)[0]) * size) >> 32 for b in range(256)], dtype=np.uint32)
    assert np.array_equal(idx[:256], want)
    assert idx.max() < size and len(np.unique(idx)) > 900
    h = np.bincount(idx // 100, minlength=10)
    assert float(((h - B / 10) ** 2 / (B / 10)).sum()) < 33.7                 # chi2, 9 dof, P ~ 1e-4
    assert not np.array_equal(idx, O.replay_sample(seed, step + 1, size, B))
