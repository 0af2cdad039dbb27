"""Test helper: random concurrent histories that are linearizable BY CONSTRUCTION, and mutators.

A global clock ticks; at each tick one random process either invokes an operation, takes
its effect on a plain Python list (the linearization point), or returns.  The effect order
is therefore a witness linearization.  No oracle code is used here.
"""
import random


def gen_history(seed, procs, n_ops, capacity, p_enq=0.5, values_from=1):
    rng = random.Random(seed)
    q = []
    t = 0
    nextval = values_from
    state = {}   # proc -> dict(op, arg, call, status, val, done)
    rows = []
    started = 0
    while started < n_ops or state:
        t += rng.randint(1, 3)
        p = rng.randrange(procs)
        s = state.get(p)
        if s is None:
            if started >= n_ops:
                continue
            started += 1
            if rng.random() < p_enq:
                state[p] = dict(op=0, arg=nextval, call=t, lin=False)
                nextval += 1
            else:
                state[p] = dict(op=1, arg=0, call=t, lin=False)
        elif not s["lin"]:
            if s["op"] == 0:
                if len(q) < capacity:
                    q.append(s["arg"]); s["status"] = 0
                else:
                    s["status"] = 1
                s["val"] = 0
            else:
                if q:
                    s["val"] = q.pop(0); s["status"] = 0
                else:
                    s["val"] = 0; s["status"] = 2
            s["lin"] = True
        else:
            rows.append((p, s["op"], s["arg"], s["status"], s["val"], s["call"], t))
            del state[p]
    return rows, list(q)


def mutate(rows, seed):
    """Returns a (possibly non-linearizable) variant: swap two dequeue results, duplicate a
    result, invent a value, or shift an interval."""
    rng = random.Random(seed)
    rows = [list(r) for r in rows]
    deqs = [i for i, r in enumerate(rows) if r[1] == 1 and r[3] == 0]
    kind = rng.randrange(4)
    if kind == 0 and len(deqs) >= 2:
        a, b = rng.sample(deqs, 2)
        rows[a][4], rows[b][4] = rows[b][4], rows[a][4]
    elif kind == 1 and len(deqs) >= 2:
        a, b = rng.sample(deqs, 2)
        rows[a][4] = rows[b][4]
    elif kind == 2 and deqs:
        rows[rng.choice(deqs)][4] = 10_000_000 + rng.randrange(100)
    else:
        i = rng.randrange(len(rows))
        d = rng.randint(1, 40)
        rows[i][5] += d
        rows[i][6] += d
    return [tuple(r) for r in rows]
