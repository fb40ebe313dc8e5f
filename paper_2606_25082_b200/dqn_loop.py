"""The paper's training loop driven through the C ABI: simulated days feed the replay ring, the tensor-core
training step learns from it, the learned network drives the next day's epsilon-greedy decisions.

Everything that computes runs in libmigsim.so: `mig_sim_step` (one decision epoch of every environment), `mig_q_eval` (the
bit-reproducible forward that picks the actions), `mig_replay_push`, `mig_dqn_train_step`, `mig_dqn_sync_target`.  This file
only sequences those calls and draws the exploration coin flips with torch's generator (device tensors, no host round trip
inside a day); it holds none of the method's arithmetic.

    python -m paper_2606_25082_b200.dqn_loop --envs 1024 --days 4
"""
from __future__ import annotations

import argparse
import dataclasses

import numpy as np
import torch

from . import binding as B
from . import workloads as W


def train(sp: W.SimParams, qnet: W.QNetWeights, n_envs: int, days: int, *, algo: int = W.ALGO_EDF_SS_R, cfg0: int = 1, seed: int = 0,
          batch: int = 4096, steps_per_epoch: int = 2, lr: float = 0.01, gamma: float = 0.9, eps0: float = 1.0, eps1: float = 0.1,
          sync_every: int = 24, log=None):
    """Runs `days` simulated days of `n_envs` environments.  Per decision epoch: epsilon-greedy action from the online network,
    one `mig_sim_step`, the transition (s, a, r, s', done) into the replay ring, `steps_per_epoch` training steps; the target
    network is synchronised every `sync_every` training steps; epsilon decays linearly from eps0 to eps1 over the days.
    Returns (trained QNetWeights, per-day dict of mean loss / mean return / mean energy / mean tardiness)."""
    assert torch.cuda.is_available(), "the training loop needs a CUDA device (no CPU fallback)"
    n_cfg = sp.n_configs
    sim = B.MigSim(sp, n_envs, seed)
    dqn = B.Dqn(qnet, replay_capacity=sp.n_epochs * n_envs * 2, batch=batch, gamma=gamma, lr=lr, seed=seed)
    d_algo = torch.full((n_envs,), algo, dtype=torch.uint8, device="cuda")
    d_cfg0 = torch.full((n_envs,), cfg0, dtype=torch.uint8, device="cuda")
    state, nxt = sim.alloc_state(), sim.alloc_state()
    reward = torch.zeros(n_envs, dtype=torch.float32, device="cuda")
    greedy = torch.zeros(n_envs, dtype=torch.uint8, device="cuda")
    loss = torch.zeros(1, dtype=torch.float32, device="cuda")
    tot = sim.alloc_totals()
    ret = torch.zeros(n_envs, dtype=torch.float32, device="cuda")
    gen = torch.Generator(device="cuda"); gen.manual_seed(seed)
    history, n_train = [], 0
    net = B.QNet(qnet)
    for day in range(days):
        eps = eps0 + (eps1 - eps0) * (day / max(1, days - 1))
        sim.reset(day, d_algo, d_cfg0, state_out=state)
        losses = []
        for k in range(sp.n_epochs):
            net.q_eval(state, argmax_out=greedy)                                   # greedy action of every environment
            explore = torch.rand(n_envs, device="cuda", generator=gen) < eps
            rnd = torch.randint(0, n_cfg, (n_envs,), device="cuda", generator=gen, dtype=torch.int64).to(torch.uint8)
            action = torch.where(explore, rnd, greedy).contiguous()
            sim.step(action, state_out=nxt, reward_out=reward)
            done = torch.full((n_envs,), 1 if k == sp.n_epochs - 1 else 0, dtype=torch.uint8, device="cuda")
            dqn.push(state, action, reward, nxt, done)
            state, nxt = nxt, state
            for _ in range(steps_per_epoch):
                dqn.train_step(n_train, loss_out=loss)
                losses.append(loss.clone())
                n_train += 1
                if n_train % sync_every == 0:
                    dqn.sync_target()
            if (k + 1) % 6 == 0 or k == sp.n_epochs - 1:                           # the acting network follows the online one
                net.close()
                net = B.QNet(dqn.weights(0))
        sim.totals(tot)
        sim.aux(return_out=ret)
        torch.cuda.synchronize()
        t = B.totals_to_numpy(tot)
        rec = {"day": day, "epsilon": eps, "loss": float(torch.stack(losses).mean().item()), "return": float(ret.mean().item()),
               "energy_mj": float(t["energy_mj"].mean()), "tardiness_s": float(t["tardiness_s"].mean()), "repartitions": float(t["n_repart"].mean())}
        history.append(rec)
        if log:
            log(rec)
    out = dqn.weights(0)
    net.close(); dqn.close(); sim.close()
    return out, history


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--envs", type=int, default=1024)
    ap.add_argument("--days", type=int, default=4)
    ap.add_argument("--batch", type=int, default=4096)
    a = ap.parse_args()
    # the paper's setting on the synthetic workload: 12 configurations + MIG disabled, whole-GPU 4 s penalty, restricted EDF-SS;
    # reward weights that put an hour of energy (~4e8 mJ) and of tardiness on the scale of 1
    sp = dataclasses.replace(W.benchmark_params(), w_energy=1e-9, w_tardy=1e-5, util_hist=0)
    qnet = W.make_qnet(1003, n_actions=sp.n_configs, hidden=256)
    train(sp, qnet, a.envs, a.days, batch=a.batch, log=lambda r: print(r, flush=True))


if __name__ == "__main__":
    main()
