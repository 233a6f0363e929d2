#!/usr/bin/env python
"""Writes the cached oracle references under tests/golden/ ("the full oracle is run once ... cached").

    python tests/golden/make_reference.py [o5_spec_cat0 o5_spec_cat1 o5_spec_cat2 o5_photo full_pop sel_heavy]

Imports only `oracle` (the fp64 CPU oracle) and `workloads` (seeded inputs); no value in the files it writes comes from
the CUDA path.  Runs on the CPU container (no GPU); the whole set takes about an hour on 8 cores.  Each file holds, for
a set of hyper-parameter points, what the oracle returns for EVERY event of the workload at full size: per-event log I,
the bandwidths, log xi, N_eff, the total log L and the flags, plus a hash of the inputs they belong to.

    python tests/golden/make_reference.py --stamp [names]

`--stamp` does not rerun the hour-long oracle job: for every existing file it recomputes a few (event, lambda) units with the
oracle as it stands, requires them to equal the stored values to 1e-12, and then records `oracle_sha256` (the hash of
oracle/chim_oracle.c and oracle/binding.py, `oracle_hash()`), which tests/test_golden_fresh.py compares with the live sources:
a later change to the oracle makes every cached file stale until it is rewritten or re-stamped by this script.

Lambda sets (`pick_lambdas`): rows of the workload's own batch (so that the GPU test can read them out of the launch
bench.py times) -- the fiducial, the first random rows, and the rows with the largest m_low, where events lose their
support (R21) -- plus the 16 corners of the (H0, Om, Xi0, n) box, which are not in the batch (index -1).
"""
import hashlib
import itertools
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import oracle as O                                      # noqa: E402
from workloads import LAMBDA_BOX, LAMBDA_NAMES, make_workload   # noqa: E402

HERE = os.path.dirname(os.path.abspath(__file__))

# name -> (config, catalog, rows of the batch taken first, rows with the largest m_low, box corners)
SETS = {
    "o5_spec_cat0": ("o5_spec", 0, 32, 16, 16),
    "o5_spec_cat1": ("o5_spec", 1, 32, 16, 16),
    "o5_spec_cat2": ("o5_spec", 2, 32, 16, 16),
    "o5_photo": ("o5_photo", 0, 12, 0, 4),
    "full_pop": ("full_pop", 0, 4, 0, 0),
    "sel_heavy": ("sel_heavy", 0, 4, 0, 0),
}


def input_hash(w):
    h = hashlib.sha256()
    for a in (w.sample_off, w.dL, w.m1d, w.m2d, w.ln_prior, w.grid_off, w.z_grid, w.p_gal, w.inj_dL, w.inj_m1d, w.inj_m2d,
              w.inj_ln_pdraw, w.lam):
        h.update(np.ascontiguousarray(a).tobytes())
    h.update(str(int(w.n_inj_total)).encode())
    return h.hexdigest()


def oracle_hash():
    """sha256 over the oracle's sources: what the cached values were computed with."""
    h = hashlib.sha256()
    for f in ("chim_oracle.c", "binding.py"):
        with open(os.path.join(ROOT, "oracle", f), "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()


def check_units(w):
    """(row of the file, event) units recomputed by --stamp and by tests/test_golden_fresh.py: first, middle and last event
    on the first, middle and last stored lambda."""
    return [(0, 0), (1, w.n_events // 2), (-1, w.n_events - 1)]


def recompute_unit(w, lam, ev):
    """log I of one event under one lambda with the oracle as it stands (same call as loglike_workload makes per event)."""
    s, g = slice(w.sample_off[ev], w.sample_off[ev + 1]), slice(w.grid_off[ev], w.grid_off[ev + 1])
    r = O.loglike_batch(lam, np.array([0, s.stop - s.start]), w.dL[s], w.m1d[s], w.m2d[s], w.ln_prior[s],
                        np.array([0, g.stop - g.start]), w.z_grid[g], w.p_gal[g])
    return float(r["event_logI"][0, 0])


def stamp(names):
    for name in names:
        cfg, cat = SETS[name][:2]
        path = os.path.join(HERE, f"ref_{name}.npz")
        g = dict(np.load(path))
        w = make_workload(cfg, catalog=cat)
        assert input_hash(w) == str(g["input_sha256"]), f"{name}: the file belongs to other inputs"
        for row, ev in check_units(w):
            got, ref = recompute_unit(w, g["lam"][row], ev), float(g["event_logI"][row, ev])
            assert (np.isnan(got) and np.isnan(ref)) or got == ref or abs(got - ref) <= 1e-12 * abs(ref), (name, row, ev, got, ref)
        g["oracle_sha256"] = oracle_hash()
        np.savez_compressed(path, **g)
        print(f"{name}: {len(check_units(w))} units recomputed, equal; stamped {g['oracle_sha256'][:16]}", flush=True)


def pick_lambdas(w, n_first, n_mlow, n_corner):
    idx = list(range(n_first))
    by_mlow = [int(i) for i in np.argsort(-w.lam[:, LAMBDA_NAMES.index("m_low")], kind="stable") if i >= n_first]
    idx += by_mlow[:n_mlow]
    lam = [w.lam[i] for i in idx]
    corners = list(itertools.product(*(LAMBDA_BOX[k] for k in ("H0", "Om", "Xi0", "n"))))
    step = max(1, len(corners) // max(n_corner, 1))
    for c in corners[::step][:n_corner]:
        v = w.fiducial.copy()
        v[:4] = c
        lam.append(v)
        idx.append(-1)
    return np.array(idx, dtype=np.int64), np.array(lam)


def main(names):
    for name in names:
        cfg, cat, n_first, n_mlow, n_corner = SETS[name]
        t0 = time.time()
        w = make_workload(cfg, catalog=cat)
        idx, lam = pick_lambdas(w, n_first, n_mlow, n_corner)
        print(f"{name}: {w.n_events} events, {w.n_det} injections, {len(idx)} lambda; inputs in {time.time() - t0:.0f} s", flush=True)
        out = {k: [] for k in ("loglike", "event_logI", "logxi", "neff", "h", "flags")}
        for i, la in enumerate(lam):
            t1 = time.time()
            r = O.loglike_workload(w, lam=la)
            for k in out:
                out[k].append(r[k][0])
            print(f"  lambda {i + 1}/{len(lam)} (batch row {idx[i]}): log L = {r['loglike'][0]:.6f}  [{time.time() - t1:.1f} s]", flush=True)
        np.savez_compressed(os.path.join(HERE, f"ref_{name}.npz"), config=cfg, catalog=cat, lam_index=idx, lam=lam,
                            input_sha256=input_hash(w), oracle_sha256=oracle_hash(), n_inj_total=int(w.n_inj_total), z_cat_max=w.z_cat_max,
                            **{k: np.array(v) for k, v in out.items()})
        print(f"{name}: written in {time.time() - t0:.0f} s", flush=True)


if __name__ == "__main__":
    if "--stamp" in sys.argv[1:]:
        stamp([a for a in sys.argv[1:] if a != "--stamp"] or list(SETS))
    else:
        main(sys.argv[1:] or list(SETS))
