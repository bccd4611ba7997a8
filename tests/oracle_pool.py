"""Test infrastructure: run the CPU oracle (oracle/nbs_oracle.py, unchanged) on several host cores.

The oracle is single-threaded numpy for most of its time.  The full-size parity tests need tier B
(`correlator_fft`) for all 52 channels on a 16^3 slice (about 5 CPU-minutes), so the channel list is
split into one task per channel and the tasks run in forked worker processes; every task calls the
oracle's own `all_blocks` + `correlator_fft` on its channel with the same propagators.  Nothing of
the method's arithmetic lives here.
"""
from __future__ import annotations

import multiprocessing as mp
import os

import numpy as np

_STATE: dict = {}


def n_workers(cap: int = 24) -> int:
    try:
        n = len(os.sched_getaffinity(0))
    except AttributeError:
        n = os.cpu_count() or 1
    return max(1, min(cap, n))


def _limit_threads():
    try:
        import threadpoolctl
        threadpoolctl.threadpool_limits(1)
    except Exception:
        pass


def _tierB_task(args):
    key, ch = args
    from oracle import nbs_oracle as O
    _limit_threads()
    L, S = _STATE[key]
    B = O.all_blocks(S, O.sink_names([ch]))
    return O.correlator_fft(L, B, [ch])[0]


def tierB_channels(cases, workers: int | None = None):
    """cases: list of (L, S, chans).  Returns, per case, F[ch, a1, a2, a3, a4, r] from the oracle's tier B, one
    forked task per (case, channel), longest channels first."""
    from oracle import nbs_oracle as O
    tasks = []
    for ic, (L, S, chans) in enumerate(cases):
        _STATE[ic] = (L, S)
        for j, ch in enumerate(chans):
            cost = L ** 3 * len(O.diagrams(ch))
            tasks.append((cost, ic, j, ch))
    tasks.sort(key=lambda t: -t[0])
    workers = workers or n_workers()
    ctx = mp.get_context("fork")  # the propagators are inherited, not pickled
    with ctx.Pool(min(workers, len(tasks))) as pool:
        res = pool.map(_tierB_task, [(ic, ch) for _, ic, _, ch in tasks], chunksize=1)
    out = []
    for ic, (L, S, chans) in enumerate(cases):
        F = np.empty((len(chans), 4, 4, 4, 4, L ** 3), dtype=np.complex128)
        for (_, jc, j, _), r in zip(tasks, res):
            if jc == ic:
                F[j] = r
        out.append(F)
    _STATE.clear()
    return out


def _momentum_task(args):
    """Oracle blocks of one baryon on a chunk of sites, projected on the sampled momenta:
    sum_x exp(-i q.x) B(x) for q in qs (the definition of the forward transform, reading A7)."""
    key, name, lo, hi = args
    from oracle import nbs_oracle as O
    _limit_threads()
    L, S, qs = _STATE[key]
    Sc = {f: S[f][lo:hi] for f in "uds"}
    B = O.block(Sc, name).reshape(hi - lo, -1)
    x = np.arange(lo, hi)
    xyz = np.stack([x % L, (x // L) % L, x // (L * L)], axis=1)
    qxyz = np.stack([qs % L, (qs // L) % L, qs // (L * L)], axis=1)
    phase = np.exp(-2j * np.pi * (qxyz @ xyz.T) / L)  # [nq, sites]
    return name, phase @ B


def blocks_at_momenta(L, S, names, qs, chunk: int = 2048, workers: int | None = None):
    """{name: B~(q) for q in qs, shape [nq, 4, 12, 12, 12]} from the oracle's x-space blocks of ALL sites, built
    chunk by chunk in forked workers (3.6 GB per baryon at 32^3 never exists at once)."""
    V = L ** 3
    _STATE["m"] = (L, S, np.asarray(qs))
    tasks = [("m", n, lo, min(V, lo + chunk)) for n in names for lo in range(0, V, chunk)]
    ctx = mp.get_context("fork")
    with ctx.Pool(min(workers or n_workers(), len(tasks))) as pool:
        res = pool.map(_momentum_task, tasks, chunksize=1)
    out = {n: np.zeros((len(qs), 4 * 1728), dtype=np.complex128) for n in names}
    for name, part in res:
        out[name] += part
    _STATE.clear()
    return {n: v.reshape(len(qs), 4, 12, 12, 12) for n, v in out.items()}
