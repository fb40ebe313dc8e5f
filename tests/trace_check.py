"""Independent replay of an event trace: conservation invariants and re-integration of energy / tardiness.

Takes only the INPUT tables (workloads.SimParams) and an event list; it does not know any scheduling rule.
Used against the oracle's traces (CPU tests) and the CUDA library's traces (GPU tests).
North-star invariants: every job finishes exactly once, slice capacities never exceeded, energy equals the
sum of per-interval power x duration.
"""
from __future__ import annotations

EV_ARRIVE, EV_DROP, EV_START, EV_PREEMPT, EV_COMPLETE, EV_CRIT, EV_SLICE_UP, EV_REPART = range(1, 9)
SIZE_IDX = {1: 0, 2: 1, 3: 2, 4: 3, 7: 4}


class TraceError(AssertionError):
    pass


def _chk(cond, msg):
    if not cond:
        raise TraceError(msg)


def replay(sp, cfg0, trace, *, jobs_in=None, truncated=False):
    event_driven = bool(getattr(sp, "decide_on_events", 0))   # reading #27: REPART may follow any arrival / completion
    """Returns dict(energy_by_epoch[list n_epochs+1], tard_by_epoch, completions{id: t}, arrivals{id: (t, cls, due)},
    n_preempt, n_start, busy_unit_s, t_last).  Raises TraceError on any violated invariant."""
    ne, es = sp.n_epochs, sp.epoch_s
    size_at = sp.size_at_slot
    cfg = int(cfg0)
    slices = {p: {"size": int(size_at[cfg][p]), "down": False, "job": None} for p in range(7) if size_at[cfg][p]}
    jobs = {}           # id -> dict(cls, due, arr, work, done, slot, t_start, completed)
    energy = [0] * (ne + 1)
    tard = [0] * (ne + 1)
    busy_us = 0
    t_prev = 0
    n_preempt = n_start = 0
    last_completion_t = 0

    def speed_on(cls, size):           # size code 8: the whole GPU with MIG disabled (reading #29)
        return int(sp.speed_nomig[cls]) if size == 8 else int(sp.speed[cls][SIZE_IDX[size]])

    def power():
        u = sum(min(s["size"], 7) for s in slices.values() if s["job"] is not None)
        _chk(u <= 7, "busy units exceed 7")
        p = int(sp.curve_mw[u])
        for s in slices.values():
            if s["size"] == 8:
                p += int(sp.p_busy_nomig_mw if s["job"] is not None else sp.p_idle_nomig_mw)
            else:
                p += int(sp.p_busy_mw[SIZE_IDX[s["size"]]] if s["job"] is not None else sp.p_idle_mw[SIZE_IDX[s["size"]]])
        return p, u

    def advance(t_to):
        """integrate over [t_prev, t_to), split at epoch boundaries (record k covers (k*es, (k+1)*es], drain after)"""
        nonlocal t_prev, busy_us
        _chk(t_to >= t_prev, "time goes backwards")
        p, u = power()
        t = t_prev
        while t < t_to:
            k = min(t // es, ne)
            seg_end = t_to if k >= ne else min(t_to, (k + 1) * es)
            energy[k] += p * (seg_end - t)
            busy_us += u * (seg_end - t)
            t = seg_end
        for s in slices.values():
            if s["job"] is not None:
                j = jobs[s["job"]]
                j["done"] += (t_to - t_prev) * speed_on(j["cls"], s["size"])
        t_prev = t_to

    def rec_index(t):
        # an event AT an epoch boundary belongs to the epoch that ends there; the prologue (REPART and what follows
        # at the same tick) belongs to the next epoch -- handled by the caller via 'after_repart'
        if t == 0:
            return 0
        return min((t - 1) // es, ne)

    after_repart_tick = None
    ambiguous = False
    for ev in trace:
        t, ty, slot, aux, job, value = int(ev["t"]), int(ev["type"]), int(ev["slot"]), int(ev["aux"]), int(ev["job"]), int(ev["value"])
        advance(t)
        if ty == EV_REPART:
            after_repart_tick = t
        k = rec_index(t)
        if after_repart_tick == t and t % es == 0 and t // es < ne:
            k = t // es
        if ty == EV_ARRIVE or ty == EV_DROP:
            _chk(job not in jobs, "job id %d arrives twice" % job)
            _chk(0 <= aux < sp.n_classes, "bad class")
            if jobs_in is not None:
                _chk(t == int(jobs_in[job]["arr"]) and value == int(jobs_in[job]["due"]), "scripted job mismatch")
            if ty == EV_DROP:
                jobs[job] = None
                continue
            jobs[job] = {"cls": aux, "due": value, "arr": t, "done": 0, "slot": None, "completed": False, "work": None}
            _chk(sum(1 for j in jobs.values() if j and not j["completed"]) <= sp.cap, "cap exceeded")
        elif ty == EV_START:
            j = jobs.get(job)
            _chk(j is not None and not j["completed"], "START of unknown/finished job")
            _chk(j["slot"] is None, "START of a job that already runs (job %d)" % job)
            _chk(slot in slices and slices[slot]["size"] == aux, "START on a non-existent slice")
            _chk(not slices[slot]["down"], "START on a down slice")
            _chk(slices[slot]["job"] is None, "START on an occupied slice")
            if j["work"] is None:
                j["work"] = value + j["done"]          # first START reveals the work; later ones must agree
            _chk(value == j["work"] - j["done"], "START rem mismatch job %d: %d vs %d" % (job, value, j["work"] - j["done"]))
            slices[slot]["job"] = job
            j["slot"] = slot
            n_start += 1
        elif ty == EV_PREEMPT:
            j = jobs.get(job)
            _chk(j is not None and j["slot"] == slot and slices[slot]["job"] == job, "PREEMPT of a job not on that slice")
            _chk(value == j["work"] - j["done"] and value > 0, "PREEMPT rem mismatch")
            slices[slot]["job"] = None
            j["slot"] = None
            n_preempt += 1
        elif ty == EV_COMPLETE:
            j = jobs.get(job)
            _chk(j is not None and j["slot"] == slot and slices[slot]["job"] == job, "COMPLETE of a job not on that slice")
            v = speed_on(j["cls"], slices[slot]["size"])
            _chk(j["work"] <= j["done"] < j["work"] + v, "work conservation: done=%d work=%d v=%d" % (j["done"], j["work"], v))
            _chk(value == max(t - j["due"], 0), "tardiness value")
            vmax = max([int(x) for x in sp.speed[j["cls"]]] + ([int(sp.speed_nomig[j["cls"]])] if getattr(sp, "speed_nomig", None) is not None else []))
            _chk(t >= j["arr"] + -(-j["work"] // vmax), "finished faster than on the fastest slice")
            tard[k] += value
            slices[slot]["job"] = None
            j["slot"] = None
            j["completed"] = True
            last_completion_t = t
        elif ty == EV_CRIT:
            j = jobs.get(job)
            _chk(j is not None and j["slot"] is None and not j["completed"], "CRIT of a non-waiting job")
            _chk(1 <= aux <= sp.crit_max, "crit count out of range")
        elif ty == EV_SLICE_UP:
            _chk(slot in slices and slices[slot]["down"], "SLICE_UP of a slice that is not down")
            slices[slot]["down"] = False
        elif ty == EV_REPART:
            old, new = aux >> 8, aux & 0xFF
            _chk(old == cfg and new != cfg and new < sp.n_configs, "REPART ids")
            _chk(event_driven or t % es == 0, "REPART off an epoch boundary")
            if event_driven and t % es == 0 and 0 < t // es < ne + 1:
                ambiguous = True       # an event-driven REPART at t_end belongs to the epoch that ends, a prologue to the next
            energy[k] += int(sp.repart_energy_mj)
            newsl = {}
            for p in range(7):
                g = int(size_at[new][p])
                if not g:
                    continue
                if p in slices and slices[p]["size"] == g and not getattr(sp, "repart_all_down", 0):
                    newsl[p] = slices[p]
                else:
                    newsl[p] = {"size": g, "down": sp.repart_downtime_s > 0, "job": None}
            for p, s in slices.items():
                if p not in newsl or newsl[p] is not s:
                    _chk(s["job"] is None, "slice destroyed while a job runs on it (no PREEMPT before REPART)")
            slices = newsl
            cfg = new
        else:
            raise TraceError("unknown event type %d" % ty)

    live = [i for i, j in jobs.items() if j and not j["completed"]]
    if not truncated:
        _chk(not live, "jobs never completed: %s" % live[:5])
        # idle power runs through the day; in the drain it stops at the last completion
        advance(max(t_prev, ne * es))
    return {"energy": energy, "tard": tard, "jobs": jobs, "n_preempt": n_preempt, "n_start": n_start,
            "ambiguous": ambiguous, "busy_unit_s": busy_us, "t_last": max(last_completion_t, ne * es) if not truncated else t_prev, "cfg_end": cfg}


def check_against_records(sp, cfg0, trace, recs, totals, **kw):
    """Replay + compare the re-integrated energy / tardiness with the per-epoch records and the totals."""
    truncated = bool(int(totals["status"]) & 1)
    out = replay(sp, cfg0, trace, truncated=truncated, **kw)
    ne = sp.n_epochs
    if not truncated and not out["ambiguous"]:
        for k in range(ne + 1):
            _chk(out["energy"][k] == int(recs[k]["energy_mj"]), "epoch %d energy %d != %d" % (k, out["energy"][k], int(recs[k]["energy_mj"])))
            _chk(out["tard"][k] == int(recs[k]["tardiness_s"]), "epoch %d tardiness" % k)
    if not truncated:
        _chk(sum(out["energy"]) == int(totals["energy_mj"]), "total energy")
        _chk(out["busy_unit_s"] == int(totals["busy_unit_s"]), "busy unit seconds")
    _chk(sum(out["tard"]) == int(totals["tardiness_s"]), "total tardiness")
    _chk(sum(int(r["energy_mj"]) for r in recs) == int(totals["energy_mj"]), "sum of epoch energies")
    _chk(sum(int(r["tardiness_s"]) for r in recs) == int(totals["tardiness_s"]), "sum of epoch tardiness")
    n_arr = sum(1 for j in out["jobs"].values())
    n_drop = sum(1 for j in out["jobs"].values() if j is None)
    n_done = sum(1 for j in out["jobs"].values() if j and j["completed"])
    _chk(n_arr == int(totals["n_jobs"]) and n_drop == int(totals["n_dropped"]) and n_done == int(totals["n_completed"]), "job counts")
    if not truncated:
        _chk(n_arr == n_done + n_drop, "arrivals != completed + dropped")
    _chk(out["n_preempt"] == int(totals["n_preempt"]) and out["n_start"] == int(totals["n_start"]), "preempt/start counts")
    _chk(len(trace) == int(totals["n_events"]), "event count")
    return out
