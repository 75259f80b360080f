"""Oracle references for the full-size registration parity tests (BASELINE.json configs 2, 3, 4).

One oracle registration of a 256x256x100 pair costs minutes of one host core (about 0.8 s per fine
iteration on the GPU box), so the references are computed in background worker processes -- each one the
oracle exactly as it stands, single-threaded -- started as soon as test collection shows that they will be
needed (tests/conftest.py), while the other GPU tests run.  Workers are spawned, not forked: the pytest
process holds a CUDA context.  Only oracle/ and the seeded input generators are imported here.

A worker walks the multi-scale driver itself (restrict, per-level single-level registrations chained through
their initial field, prolong: the composition that tests/test_oracle_pins.py::test_multilevel_driver_wiring
pins bit for bit against oracle_register) so that it can keep PROBES along the way: the state before and
after PROBE_LEN iterations at a few points of the trajectory.  The registrations of these hard-edged noisy
phantoms amplify rounding differences (the oracle differs from itself by 0.05 voxel after 25 iterations when
the moving image moves by one ulp), so the end state of a 300-iteration run can only be compared
statistically; a probe re-synchronises the CUDA path with the oracle's state and compares the next few
iterations at the per-kernel tolerance.  `*_M1ulp` cases are the oracle against itself with every voxel of M
moved by one ulp: the conditioning of the problem, measured without the CUDA path.
"""
from __future__ import annotations

import concurrent.futures as cf
import multiprocessing as mp
import os
import tempfile

import numpy as np

# name -> (dims, phantom seed, variant, alpha, iterations per level coarse -> fine)
BASE_CASES = {
    "config2_passive": ((256, 256, 100), 202, 0, 1.0, [300]),
    "config3_active": ((256, 256, 100), 202, 2, 1.0, [100, 100, 100]),
    "config3_double": ((256, 256, 100), 202, 3, 1.0, [100, 100, 100]),
    "config3_adjusted_a0.4": ((256, 256, 100), 202, 4, 0.4, [100, 100, 100]),
    "config4_inverse_consistent": ((256, 256, 110), 404, 5, 1.0, [100, 100, 100]),
}
# well-conditioned pairs (phantoms.textured_pair: intensity gradient almost everywhere, no flat regions): the end state
# is held to the plain 1e-2 voxel bar of north_star, no conditioning measurement needed
TEXTURED_CASES = {
    "textured_config2_passive": ((256, 256, 100), 212, 0, 1.0, [300]),
    "textured_config3_double": ((256, 256, 100), 212, 3, 1.0, [100, 100, 100]),
}
FULL_CASES = dict(BASE_CASES)
FULL_CASES.update({n + "_M1ulp": v for n, v in BASE_CASES.items()})
FULL_CASES.update(TEXTURED_CASES)
PROBE_LEN = 5
# A host with few cores cannot run the references side by side in a few minutes: the counts are cut
# (full sizes kept) and the tests say so.
REDUCED_ITERS = {1: [40], 3: [30, 30, 30]}


def iterations_for(name):
    iters = FULL_CASES[name][4]
    if (os.cpu_count() or 1) < 10:
        return REDUCED_ITERS[len(iters)]
    return iters


def probe_points(n_iters):
    """Iterations at which a probe starts on a level of n_iters iterations: start, middle, end."""
    pts = sorted({0, (n_iters // 2 // PROBE_LEN) * PROBE_LEN, ((n_iters - PROBE_LEN) // PROBE_LEN) * PROBE_LEN})
    return [q for q in pts if 0 <= q and q + PROBE_LEN <= n_iters]


def perturb_one_ulp(vol, seed=99):
    """Every voxel moved to the next float32 up or down (seeded coin per voxel)."""
    sgn = np.random.default_rng(seed).integers(0, 2, vol.shape).astype(np.float32) * 2 - 1
    return np.nextafter(vol, vol + sgn).astype(np.float32)


def chained_register(O, variant, alpha, S, M, iters, probes=True):
    """The multi-scale driver walked level by level and segment by segment (same trajectory as
    O.register(variant, alpha, 1.0, S, M, iters), bit for bit), keeping the probes."""
    levels = len(iters)
    ic = variant == 5
    Sl, Ml = [S], [M]
    for _ in range(1, levels):
        Sl.append(O.restrict(Sl[-1]))
        Ml.append(O.restrict(Ml[-1]))
    u = np.zeros((3,) + Sl[-1].shape, np.float32)
    out = {}
    stats = []
    for step in range(levels):
        l = levels - 1 - step
        pts = probe_points(iters[step]) if probes else []
        n = 0
        while n < iters[step]:
            if n in pts:
                seg = PROBE_LEN
            else:
                nxt = [q for q in pts if q > n]
                seg = (nxt[0] if nxt else iters[step]) - n
            r = O.register(variant, alpha, 1.0, Sl[l], Ml[l], [seg], u0=u, ub0=-u if ic else None)
            if n in pts:
                out[f"probe_L{l}_n{n}_before"] = u
                out[f"probe_L{l}_n{n}_after"] = r["u"]
                out[f"probe_L{l}_n{n}_stats"] = r["stats"]
            if ic:
                assert np.array_equal(r["ub"], -r["u"])      # pin P10 along the whole trajectory
            u = r["u"]
            stats.append(r["stats"])
            n += seg
        if l > 0:
            u = O.prolong(u, Sl[l - 1].shape)
    out["u"] = u
    out["stats"] = np.concatenate(stats)
    return out


def _worker(name, out_dir):
    from oracle import oracle as O
    from paper_0909_0928_b200 import phantoms as P
    dims, seed, variant, alpha, _ = FULL_CASES[name]
    textured = name in TEXTURED_CASES
    S, M, _truth = P.textured_pair(dims, seed) if textured else P.lung_pair(dims, seed)
    perturbed = name.endswith("_M1ulp")
    if perturbed:
        M = perturb_one_ulp(M)
    out = chained_register(O, variant, alpha, S, M, iterations_for(name), probes=not (perturbed or textured))
    ic = variant == 5
    out["final_ssd"] = O.final_ssd(variant, S, M, out["u"], -out["u"] if ic else None)
    if ic:
        out["ic_mean"], out["ic_max"] = O.ic_error(out["u"], -out["u"])
    path = os.path.join(out_dir, name + ".npz")
    np.savez(path, **out)
    return path


class FullRefs:
    """Starts every reference at construction; get(name) blocks until that one is there."""

    def __init__(self):
        from oracle import oracle as O
        O.build()  # once, before the workers race to build it
        self.dir = tempfile.mkdtemp(prefix="demons_full_refs_")
        workers = max(1, min(len(FULL_CASES), (os.cpu_count() or 1) - 1))
        self.pool = cf.ProcessPoolExecutor(max_workers=workers, mp_context=mp.get_context("spawn"))
        # longest first
        order = sorted(FULL_CASES, key=lambda n: (not n.startswith("config4"), "config2" not in n, n))
        self.futures = {n: self.pool.submit(_worker, n, self.dir) for n in order}

    def get(self, name):
        return np.load(self.futures[name].result())

    def close(self):
        self.pool.shutdown(wait=False, cancel_futures=True)
        for f in os.listdir(self.dir):
            os.remove(os.path.join(self.dir, f))
        os.rmdir(self.dir)
