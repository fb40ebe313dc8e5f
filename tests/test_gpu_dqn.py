"""GPU parity of the DQN training step: mig_dqn_* through the C ABI (tensor-core products, 3 x TF32) vs
the double-precision oracle (oracle/dqn_oracle.c), element by element.

Tolerance ("dqn"): the products are fp32-accurate (3 x TF32 split, fp32 accumulation), the oracle is
double; every compared quantity must agree within 1e-4 of its own scale (north_star's bound for Q-values): Q-values
relative to max |Q|, the loss relatively, weights after k steps within 1e-4 of the distance they have moved plus the fp32
storage of the weights themselves (k roundings of 2^-24 |w|: the library keeps fp32 master weights, the oracle doubles).
"""
import numpy as np
import pytest
import torch

from oracle import oracle as O
from paper_2606_25082_b200 import workloads as W

pytestmark = pytest.mark.gpu

B = None
TOL = 1e-4


@pytest.fixture(scope="module", autouse=True)
def _binding():
    global B
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2606_25082_b200 import binding
    B = binding
    yield


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def make_batch(seed, n, A=12, scale=1.0):
    rng = np.random.default_rng(seed)
    s = (rng.normal(0, 1, (n, 64)) * scale).astype(np.float32)
    s2 = (rng.normal(0, 1, (n, 64)) * scale).astype(np.float32)
    a = rng.integers(0, A, n).astype(np.uint8)
    r = rng.normal(0, 1, n).astype(np.float32)
    done = (rng.random(n) < 0.25).astype(np.uint8)
    return s, a, r, s2, done


def flat(qw):
    return np.concatenate([np.asarray(x, np.float64).ravel() for x in (qw.W1, qw.b1, qw.W2, qw.b2, qw.W3, qw.b3)])


@pytest.mark.parametrize("hidden,n,A", [(256, 128, 12), (256, 1000, 12), (128, 384, 5), (256, 4096, 16)])
def test_tensor_core_forward_matches_double(hidden, n, A):
    net = W.make_qnet(21, n_actions=A, hidden=hidden)
    batch = ((n + 127) // 128) * 128
    d = B.Dqn(net, 256, batch, 0.9, 0.01, 1)
    s = make_batch(22, n, A)[0]
    q = d.q(dev(s)).cpu().numpy()
    want = O.Dqn(net, 0.9, 0.01).q(s)
    assert np.abs(q - want).max() <= TOL * np.abs(want).max(), np.abs(q - want).max() / np.abs(want).max()
    # far tighter than single-pass TF32 (2^-11 per operand): the split recovers fp32
    assert np.abs(q - want).max() <= 2e-6 * np.abs(want).max() * np.sqrt(hidden)
    # and the same numbers as the bit-reproducible FFMA forward up to fp32 rounding
    qn = B.QNet(net)
    q2 = torch.empty((n, A), dtype=torch.float32, device="cuda")
    qn.q_eval(dev(s), q_out=q2)
    assert np.abs(q - q2.cpu().numpy()).max() <= 1e-5 * np.abs(want).max()
    d.close(); qn.close()


@pytest.mark.parametrize("hidden,batch,A,steps", [(256, 128, 12, 3), (256, 1024, 12, 4), (128, 512, 7, 3), (256, 8192, 12, 2), (256, 4224, 12, 2), (128, 896, 16, 2)])
def test_training_steps_match_the_oracle(hidden, batch, A, steps):
    net = W.make_qnet(31, n_actions=A, hidden=hidden)
    gamma, lr = 0.9, 0.05
    d = B.Dqn(net, 16, batch, gamma, lr, 1)
    o = O.Dqn(net, gamma, lr)
    theta0 = o.params()
    loss_g = torch.zeros(1, dtype=torch.float32, device="cuda")
    for k in range(steps):
        s, a, r, s2, done = make_batch(40 + k, batch, A)
        if k == steps - 1:
            d.sync_target(); o.sync_target()                   # the last step runs against a target that differs from the initial one
        d.train_on(dev(s), dev(a), dev(r), dev(s2), dev(done), loss_out=loss_g)
        lo = o.train_step(s, a, r, s2, done)
        assert abs(float(loss_g.item()) - lo) <= TOL * lo, (k, float(loss_g.item()), lo)
    got, want = flat(d.weights(0)), o.params()
    moved = np.abs(want - theta0).max()
    assert moved > 1e-4
    err = np.abs(got - want).max()
    store = steps * 2.0 ** -23 * np.abs(want).max()           # the library keeps fp32 weights: one rounding of |w| per step
    assert err <= TOL * moved + store, (err, moved)
    # per tensor: each one moved, each one agrees (within 1e-4 of its own movement + the fp32 storage of its own magnitude)
    for g_, w_, t0 in zip(o.split(got), o.split(want), o.split(theta0)):
        assert np.abs(w_ - t0).max() > 0
        assert np.abs(g_ - w_).max() <= TOL * np.abs(w_ - t0).max() + steps * 2.0 ** -23 * np.abs(w_).max(), (np.abs(g_ - w_).max(), np.abs(w_ - t0).max())
    # the target network holds what the sync copied: the online weights as they were before the last step
    tg = flat(d.weights(1))
    assert np.abs(tg - o.params(1)).max() <= TOL * moved and np.abs(tg - got).max() > 0
    d.close()


@pytest.mark.parametrize("bn", ["128", "256"])
def test_both_tile_widths_of_the_hidden_layer_products(bn, monkeypatch):
    # products with N = 256 run as 128 x 256 tiles from batch 32768 on (MIG_DQN_BN overrides the rule at create): same results
    monkeypatch.setenv("MIG_DQN_BN", bn)
    test_training_steps_match_the_oracle(256, 1024, 12, 3)
    test_tensor_core_forward_matches_double(256, 1000, 12)
    monkeypatch.delenv("MIG_DQN_BN")
    net = W.make_qnet(21, n_actions=12, hidden=256)            # the rule itself: a batch of 32768 takes the wide tiles
    d = B.Dqn(net, 256, 32768, 0.9, 0.01, 1)
    s = make_batch(23, 32768, 12)[0]
    q = d.q(dev(s)).cpu().numpy()
    want = O.Dqn(net, 0.9, 0.01).q(s)
    assert np.abs(q - want).max() <= TOL * np.abs(want).max()
    d.close()


def test_k_major_weight_gradient_path_gives_the_same_step(monkeypatch):
    # MIG_DQN_MN=0 at create: every activation also written transposed, K-major weight-gradient products over the copies, bias
    # gradients as row sums (the path before the MN-major operands; kept for A/B timing).  Same oracle, same tolerance.
    monkeypatch.setenv("MIG_DQN_MN", "0")
    test_training_steps_match_the_oracle(256, 1024, 12, 3)
    test_training_steps_match_the_oracle(128, 896, 16, 2)


def test_replay_ring_and_sampling():
    A, batch, cap = 12, 256, 1000
    net = W.make_qnet(51, n_actions=A, hidden=256)
    gamma, lr, seed = 0.95, 0.02, 0x123456789A
    d = B.Dqn(net, cap, batch, gamma, lr, seed)
    o = O.Dqn(net, gamma, lr)
    ring = {k: None for k in "s a r s2 done".split()}
    host = dict(s=np.zeros((cap, 64), np.float32), a=np.zeros(cap, np.uint8), r=np.zeros(cap, np.float32), s2=np.zeros((cap, 64), np.float32),
                done=np.zeros(cap, np.uint8))
    head = size = 0
    loss_g = torch.zeros(1, dtype=torch.float32, device="cuda")
    with pytest.raises(B.MigError):
        d.train_step(0)                                        # empty ring
    for it, n in enumerate((300, 500, 450, 1700)):             # the third push wraps, the fourth is larger than the ring
        s, a, r, s2, done = make_batch(60 + it, n, A)
        d.push(dev(s), dev(a), dev(r), dev(s2), dev(done) if it != 1 else None)
        if it == 1:
            done = np.zeros(n, np.uint8)
        for i in range(n):                                     # the ring's definition: transition i -> slot (head + i) mod cap
            p = (head + i) % cap
            host["s"][p], host["a"][p], host["r"][p], host["s2"][p], host["done"][p] = s[i], a[i], r[i], s2[i], done[i]
        head = (head + n) % cap; size = min(cap, size + n)
        assert d.replay_size() == size
        idx = O.replay_sample(seed, it, size, batch)
        d.train_step(it, loss_out=loss_g)
        lo = o.train_step(host["s"][idx], host["a"][idx], host["r"][idx], host["s2"][idx], host["done"][idx])
        assert abs(float(loss_g.item()) - lo) <= TOL * lo, (it, float(loss_g.item()), lo)
    got, want = flat(d.weights(0)), o.params()
    moved = np.abs(want - flat(net)).max()
    assert np.abs(got - want).max() <= TOL * moved
    d.close()


def test_training_from_simulated_transitions_improves_the_td_error():
    # the paper's loop in small: mig_sim_step feeds the replay ring (state, action, reward, next state), the tensor-core
    # step trains on it, and the trained weights drive the next day's epsilon-greedy rollout through mig_q_eval
    n = 256
    wl = W.config_c4(n)
    import dataclasses
    sp = dataclasses.replace(wl.params, w_energy=1e-9, w_tardy=1e-5)       # rewards of order 1 (an hour of a GPU is ~4e8 mJ)
    sim = B.MigSim(sp, n, wl.seed)
    d = B.Dqn(wl.qnet, 24 * n, 1024, 0.9, 0.02, 7)
    state = sim.alloc_state(); nxt = sim.alloc_state()
    rew = torch.zeros(n, dtype=torch.float32, device="cuda")
    rng = np.random.default_rng(3)
    sim.reset(0, dev(wl.algo), dev(wl.cfg0), state_out=state)
    for k in range(24):
        act = dev(rng.integers(0, 12, n).astype(np.uint8))
        sim.step(act, state_out=nxt, reward_out=rew)
        done = torch.full((n,), 1 if k == 23 else 0, dtype=torch.uint8, device="cuda")
        d.push(state, act, rew, nxt, done)
        state, nxt = nxt, state
    assert d.replay_size() == 24 * n
    loss = torch.zeros(1, dtype=torch.float32, device="cuda")
    losses = []
    for k in range(40):
        d.train_step(k % 4, loss_out=loss)                     # four fixed batches, revisited
        losses.append(float(loss.item()))
    assert np.isfinite(losses).all() and np.mean(losses[-4:]) < np.mean(losses[:4])
    qn = B.QNet(d.weights(0))                                  # the trained network drives a rollout
    recs, tot = sim.alloc_recs(), sim.alloc_totals()
    sim.reset(1, dev(wl.algo), dev(wl.cfg0))
    sim.rollout(W.POLICY_DQN, qnet=qn, epsilon=0.1, recs_out=recs, totals_out=tot)
    torch.cuda.synchronize()
    assert int(B.totals_to_numpy(tot)["n_completed"].sum()) > 0
    sim.close(); d.close(); qn.close()


def test_boundary_errors():
    net = W.make_qnet(1, n_actions=12, hidden=256)
    for kw in (dict(batch=100), dict(batch=0), dict(replay_capacity=0), dict(gamma=1.5), dict(lr=-1.0)):
        args = dict(replay_capacity=64, batch=128, gamma=0.9, lr=0.1, seed=1); args.update(kw)
        with pytest.raises(B.MigError) as ei:
            B.Dqn(net, **args)
        assert ei.value.code == B.MIG_EINVAL
    with pytest.raises(B.MigError):
        B.Dqn(W.make_qnet(1, n_actions=12, hidden=64), 64, 128, 0.9, 0.1, 1)          # hidden must be 128 or 256
    d = B.Dqn(net, 64, 128, 0.9, 0.1, 1)
    with pytest.raises(B.MigError):
        d.q(torch.zeros((256, 64), dtype=torch.float32, device="cuda"))               # more rows than the batch
    d.close()


def test_training_loop_runs_end_to_end():
    # paper_2606_25082_b200/dqn_loop.py: simulated days -> replay ring -> tensor-core training -> the next day's decisions
    import dataclasses
    from paper_2606_25082_b200 import dqn_loop
    sp = dataclasses.replace(W.benchmark_params(jobs_per_day=600.0), w_energy=1e-9, w_tardy=1e-5, util_hist=0)
    net0 = W.make_qnet(77, n_actions=sp.n_configs, hidden=128)
    net1, hist = dqn_loop.train(sp, net0, 256, 2, batch=1024, steps_per_epoch=1, lr=0.01)
    assert len(hist) == 2 and all(np.isfinite(list(h.values())).all() for h in hist)
    assert hist[0]["repartitions"] > 1 and hist[0]["energy_mj"] > 0
    assert np.abs(flat(net1) - flat(net0)).max() > 1e-5
