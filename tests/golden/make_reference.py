#!/usr/bin/env python
"""Writes the cached oracle references under tests/golden/ ("the full oracle is run once ... cached").

    python tests/golden/make_reference.py [o5_spec_cat0 o5_spec_cat1 o5_spec_cat2 o5_photo full_pop sel_heavy]

Imports only `oracle` (the fp64 CPU oracle) and `workloads` (seeded inputs); no value in the files it writes comes from
the CUDA path.  Runs on the CPU container (no GPU); the whole set takes about an hour on 8 cores.  Each file holds, for
a set of hyper-parameter points, what the oracle returns for EVERY event of the workload at full size: per-event log I,
the bandwidths, log xi, N_eff, the total log L and the flags, plus a hash of the inputs they belong to.

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
                            input_sha256=input_hash(w), n_inj_total=int(w.n_inj_total), z_cat_max=w.z_cat_max,
                            **{k: np.array(v) for k, v in out.items()})
        print(f"{name}: written in {time.time() - t0:.0f} s", flush=True)


if __name__ == "__main__":
    main(sys.argv[1:] or list(SETS))
