"""MicSA driver loop of the oracle -- TEST INFRASTRUCTURE ONLY.

Follows the procedure of PAPER.md:208-217 (Sec. 2.8.1) with gamma = 1 daemon
per spin and an explicit list of (T, n_sweeps) steps instead of the 2^s
schedule (PAPER.md:190-192 allows any refresh times; readings R3,
R12):

    for k, (T_k, n_k, every_k) in enumerate(schedule):
        refresh all demons from Eq. (11) at T_k, Philox step index step0 + k
        for j in 1..n_k:
            sweep (even sites, then odd sites)
            if every_k > 0 and j % every_k == 0: measure
"""
from __future__ import annotations

import numpy as np

from . import measure, refresh, refresh_alpha, sweep, timesteps_walkers, wander

# PAPER.md:204 Eq. (13): walker family alpha -> (axis, direction)
EQ13 = [(0, +1), (1, +1), (2, +1), (0, -1), (1, -1), (2, -1)]


def anneal(L, s, m, J, seed, schedule, step0=0, sample_offset=0, walkers=False, t0=0):
    """Run the schedule in place on (s, m).  Returns a dict with the exact
    integer sums of every measurement row and the running minimum of E/N.
    walkers=True: one forward-X walker per spin instead of a daemon -- after
    every sweep the wandering half-cycle of parity t mod 2 (PAPER.md:200,
    :215), t = t0 + sweeps done; a refresh does not reset t.
    gamma daemons per spin: m has shape [gamma, ns, nr, N]; a
    timestep is gamma sweeps, the alpha-th one uses m[alpha]; n_sweeps and
    `every` then count timesteps, E_daemon sums over the families.  With
    walkers, family alpha wanders along Eq. (13)'s alpha-th direction after the
    gamma sweeps of a timestep (the paper uses all six with gamma = 6; for
    2 <= gamma < 6 the first gamma rows are taken, R17)."""
    ns, nr, N = s.shape
    gamma = m.shape[0] if m.ndim == 4 else 1
    assert gamma <= 6
    rows = {"sweep": [], "T": [], "E": [], "Edem": [], "Q": []}
    min_e = np.full(ns * nr, np.inf)
    t = 0
    for k, (T, n_sweeps, every) in enumerate(schedule):
        if gamma > 1:
            for alpha in range(gamma):
                refresh_alpha(L, m[alpha], seed, T, step0 + k, alpha, sample_offset)
        else:
            refresh(L, m, seed, T, step0 + k, sample_offset)
        for j in range(1, n_sweeps + 1):
            if gamma > 1:
                for alpha in range(gamma):
                    sweep(L, s, m[alpha], J, 1)
                if walkers:      # after the gamma sweeps every family wanders its own way (Eq. 13)
                    for alpha in range(gamma):
                        wander(L, m[alpha], EQ13[alpha][0], EQ13[alpha][1], (t0 + t) & 1)
            elif walkers:
                timesteps_walkers(L, s, m, J, 1, t0 + t)
            else:
                sweep(L, s, m, J, 1)
            t += 1
            if every > 0 and j % every == 0:
                if gamma > 1:
                    E, Ed, Q = measure(L, s, m[0], J)
                    Ed = sum(measure(L, s, m[alpha], J)[1] for alpha in range(gamma))
                else:
                    E, Ed, Q = measure(L, s, m, J)
                rows["sweep"].append(t)
                rows["T"].append(T)
                rows["E"].append(E)
                rows["Edem"].append(Ed)
                rows["Q"].append(Q)
                min_e = np.minimum(min_e, E / float(N))
    out = {k: np.array(v) for k, v in rows.items()}
    out["min_energy"] = min_e
    return out
