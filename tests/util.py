"""Small helpers shared by the test modules (input construction only)."""
from __future__ import annotations

import json
import os

import numpy as np

from paper_2606_25082_b200 import workloads as W

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")
LINEAR = W.speed_linear()                 # {120,240,360,480,840}
SUB05 = W.speed_sublinear(0.5)            # {317,449,550,635,840}
CAP3 = W.speed_capped(3)                  # {280,560,840,840,840}
EV_NAMES = {1: "ARRIVE", 2: "DROP", 3: "START", 4: "PREEMPT", 5: "COMPLETE", 6: "CRIT", 7: "SLICE_UP", 8: "REPART"}


def golden(name):
    with open(os.path.join(GOLDEN, name)) as f:
        return json.load(f)


def tiny_params(speeds=(LINEAR,), **kw):
    """Scripted-job parameter set: tables that the generator would use are present but irrelevant."""
    speeds = list(speeds)
    return W.make_params(speeds, [W.dur_constant(10)] * len(speeds), [1] * len(speeds),
                         jobs_per_day=200, amplitude=0.0, **kw)


def completions(trace):
    return {int(ev["job"]): int(ev["t"]) for ev in trace if ev["type"] == 5}


def events_at(trace, t):
    return [(EV_NAMES[int(ev["type"])], int(ev["job"]), int(ev["slot"])) for ev in trace if ev["t"] == t]


def cfg_idle_mw(sp, cfg):
    return int(sum(int(sp.p_idle_mw[W.SIZE_INDEX[int(g)]]) for g in sp.size_at_slot[cfg] if g))


def trace_tuple(trace):
    return [tuple(int(x) for x in ev) for ev in trace]
