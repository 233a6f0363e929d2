"""Seeded synthetic workloads shaped like BASELINE.json's five configs.

This module only *draws inputs* (PE samples, redshift grids, p_gal arrays,
hyper-parameter batches, injection sets).  It computes none of the method's
outputs and is imported by neither `oracle/` nor the CUDA library: tests,
`bench.py` and `__graft_entry__.smoke()` call it and hand the same arrays to
both sides.  The arithmetic in here (a fine cumulative-trapezoid distance
table, inverse-CDF draws) exists to give the inputs the paper's shapes and
distributions (sec. 3); its accuracy is
irrelevant to parity because both sides see the resulting numbers as data.

The paper's own inputs (MICEv2 galaxies, GWFAST PE chains, the 2x10^7
injection set) are not in the container; these workloads stand in for them.
"""
from __future__ import annotations

import dataclasses
from typing import Dict, Optional

import numpy as np

C_KMS = 299792.458

LAMBDA_NAMES = ("H0", "Om", "Xi0", "n", "alpha", "beta", "delta_m", "m_low",
                "m_high", "mu_g", "sigma_g", "lambda_g", "gamma", "kappa", "z_p")
N_LAMBDA_PARAMS = len(LAMBDA_NAMES)

# Table 1 with BASELINE.json's Om, n and m_low (R11).
FIDUCIAL = dict(H0=70.0, Om=0.3, Xi0=1.0, n=1.9, alpha=3.4, beta=1.1, delta_m=4.8,
                m_low=5.1, m_high=87.0, mu_g=34.0, sigma_g=3.6, lambda_g=0.039,
                gamma=2.7, kappa=3.0, z_p=2.0)

LAMBDA_BOX = dict(H0=(60.0, 80.0), Om=(0.2, 0.4), Xi0=(0.5, 2.0), n=(0.5, 3.0))

# name -> (config_index, n_events, n_samples, n_grid, n_gal, sigma_z, n_lambda, n_det)
CONFIGS = {
    "tiny":      dict(index=0, n_events=10,   n_samples=1000, n_grid=200,  n_gal=50,
                      sigma_z=0.001, n_lambda=1,    n_det=None, n_inj_draw=10_000),
    "o5_spec":   dict(index=1, n_events=300,  n_samples=5000, n_grid=1000, n_gal=500,
                      sigma_z=0.001, n_lambda=1024, n_det=1_000_000),
    "o5_photo":  dict(index=2, n_events=300,  n_samples=5000, n_grid=4096, n_gal=2000,
                      sigma_z=0.03,  n_lambda=1024, n_det=1_000_000),
    "full_pop":  dict(index=3, n_events=5000, n_samples=4096, n_grid=512,  n_gal=500,
                      sigma_z=0.001, n_lambda=256,  n_det=1_000_000),
    "sel_heavy": dict(index=4, n_events=300,  n_samples=5000, n_grid=1000, n_gal=500,
                      sigma_z=0.001, n_lambda=4096, n_det=10_000_000),
}
XI0_CATALOGS = (1.0, 0.6, 1.8)       # catalog_index 0, 1, 2 (O5 configs)
Z_EVENT_MAX = 1.5                    # events drawn on [0, 1.5]; also z_cat_max of the selection term
INJ_DL_RANGE = (100.0, 20000.0)
INJ_M_RANGE = (5.0, 100.0)


def lambda_vector(**over) -> np.ndarray:
    d = dict(FIDUCIAL)
    d.update(over)
    return np.array([d[k] for k in LAMBDA_NAMES], dtype=np.float64)


# ----------------------------------------------------------------------------
# generator-private cosmology / population helpers (inputs only)
# ----------------------------------------------------------------------------
class _Cosmo:
    """Fine-table flat LCDM + Xi(z) used only to place synthetic events."""

    def __init__(self, H0, Om, Xi0, n, z_max=12.0, n_tab=240_001):
        self.z = np.linspace(0.0, z_max, n_tab)
        inv_e = 1.0 / np.sqrt(Om * (1 + self.z) ** 3 + 1 - Om)
        dz = self.z[1] - self.z[0]
        dc = np.concatenate(([0.0], np.cumsum(0.5 * (inv_e[1:] + inv_e[:-1]) * dz)))
        self.dc = dc * C_KMS / H0
        self.dvdz = self.dc ** 2 * inv_e          # prop. to dV_c/dz
        xi = Xi0 + (1 - Xi0) / (1 + self.z) ** n
        self.dl = xi * (1 + self.z) * self.dc

    def dl_of_z(self, z):
        return np.interp(z, self.z, self.dl)

    def z_of_dl(self, dl):
        return np.interp(dl, self.dl, self.z)


def _psi(z, gamma, kappa, z_p):
    return (1 + z) ** gamma / (1 + ((1 + z) / (1 + z_p)) ** (gamma + kappa))


def _smooth(m, m_low, delta_m):
    mp = np.clip(m - m_low, 1e-300, None)
    with np.errstate(over="ignore", divide="ignore"):
        f = delta_m / mp + delta_m / (mp - delta_m)
        s = 1.0 / (1.0 + np.exp(f))
    s = np.where(m <= m_low, 0.0, s)
    return np.where(m >= m_low + delta_m, 1.0, s)


def _inv_cdf_draw(rng, x, pdf, size):
    cdf = np.concatenate(([0.0], np.cumsum(0.5 * (pdf[1:] + pdf[:-1]) * np.diff(x))))
    cdf /= cdf[-1]
    return np.interp(rng.random(size), cdf, x)


def _draw_source_masses(rng, n, p):
    """(m1, m2) from the fiducial power law + peak."""
    m = np.linspace(p["m_low"], 2.0 * p["m_high"], 40_001)
    pl = np.where(m <= p["m_high"], m ** (-p["alpha"]), 0.0)
    pl /= np.trapezoid(pl, m)
    g = np.exp(-0.5 * ((m - p["mu_g"]) / p["sigma_g"]) ** 2) / (p["sigma_g"] * np.sqrt(2 * np.pi))
    s = _smooth(m, p["m_low"], p["delta_m"])
    pdf1 = ((1 - p["lambda_g"]) * pl + p["lambda_g"] * g) * s
    m1 = _inv_cdf_draw(rng, m, pdf1, n)
    pdf2 = m ** p["beta"] * s
    cdf2 = np.concatenate(([0.0], np.cumsum(0.5 * (pdf2[1:] + pdf2[:-1]) * np.diff(m))))
    c_at_m1 = np.interp(m1, m, cdf2)
    m2 = np.interp(rng.random(n) * c_at_m1, cdf2, m)
    m2 = np.minimum(np.maximum(m2, p["m_low"] * (1 + 1e-9)), m1)
    return m1, m2


# ----------------------------------------------------------------------------
@dataclasses.dataclass
class Workload:
    name: str
    seed: int
    fiducial: np.ndarray            # [15]
    # events (ragged in general; these generators make them rectangular)
    sample_off: np.ndarray          # int64 [n_events+1]
    dL: np.ndarray                  # f64 [sum N_s]  Mpc
    m1d: np.ndarray                 # f64, detector-frame, m1d >= m2d
    m2d: np.ndarray
    ln_prior: np.ndarray            # ln pi(theta^d_j)
    grid_off: np.ndarray            # int64 [n_events+1]
    z_grid: np.ndarray              # f64 [sum N_z]
    p_gal: np.ndarray               # f64 [sum N_z]
    z_true: np.ndarray              # f64 [n_events] (diagnostic)
    # hyper-parameters
    lam: np.ndarray                 # f64 [n_lambda, 15]
    # injections (detected set)
    inj_dL: np.ndarray
    inj_m1d: np.ndarray
    inj_m2d: np.ndarray
    inj_ln_pdraw: np.ndarray
    n_inj_total: int
    z_cat_max: float = Z_EVENT_MAX
    meta: Optional[Dict] = None
    # "many-1d" kernel: the entries above are (event, pixel) sub-events; physical event g owns the
    # sub-events [group_off[g], group_off[g+1]) and ln_factor[k] = ln of the hyperparameter-independent pixel factor
    group_off: Optional[np.ndarray] = None
    ln_factor: Optional[np.ndarray] = None

    @property
    def n_events(self):
        return len(self.sample_off) - 1

    @property
    def n_lambda(self):
        return self.lam.shape[0]

    @property
    def n_det(self):
        return len(self.inj_dL)

    def dense_pairs(self):
        ns = np.diff(self.sample_off)
        nz = np.diff(self.grid_off)
        return int(np.sum(ns * nz)) * self.n_lambda


def draw_lambda_batch(rng, n_lambda, fid: Dict, box=LAMBDA_BOX) -> np.ndarray:
    """lam[0] = fiducial; the rest uniform in the (H0, Om, Xi0, n) box with the 11
    population parameters jittered by U(0.9, 1.1) (BASELINE.json configs)."""
    lam = np.empty((n_lambda, N_LAMBDA_PARAMS))
    fidv = np.array([fid[k] for k in LAMBDA_NAMES])
    u = rng.random((n_lambda, N_LAMBDA_PARAMS))
    for c, k in enumerate(LAMBDA_NAMES):
        if k in box:
            lo, hi = box[k]
            lam[:, c] = lo + (hi - lo) * u[:, c]
        else:
            lam[:, c] = fidv[c] * (0.9 + 0.2 * u[:, c])
    lam[0] = fidv
    return lam


def draw_injections(rng, n_det=None, n_draw=None, chunk=2_000_000):
    """Detected injections from the reference pdf + SNR proxy.

    Either keep drawing until `n_det` pass (n_inj_total = draws used), or draw
    exactly `n_draw` and keep what passes."""
    dl_lo, dl_hi = INJ_DL_RANGE
    m_lo, m_hi = INJ_M_RANGE
    keep = {k: [] for k in ("dL", "m1d", "m2d", "lnp")}
    got, drawn = 0, 0
    while True:
        n = chunk if n_draw is None else min(chunk, n_draw - drawn)
        if n <= 0:
            break
        dl = dl_lo * (dl_hi / dl_lo) ** rng.random(n)
        # m1d ~ m^-2 on [m_lo, m_hi]: inverse cdf
        u = rng.random(n)
        m1 = 1.0 / (1.0 / m_lo - u * (1.0 / m_lo - 1.0 / m_hi))
        m2 = m_lo + (m1 - m_lo) * rng.random(n)
        theta = 0.2 + 0.8 * rng.random(n)
        mc = (m1 * m2) ** 0.6 / (m1 + m2) ** 0.2
        rho = 20.0 * (mc / 26.0) ** (5.0 / 6.0) * (3000.0 / dl) * theta
        det = (rho > 20.0) & (m1 - m_lo > 1e-6)
        idx = np.flatnonzero(det)
        if n_det is not None and got + len(idx) >= n_det:
            idx = idx[: n_det - got]
            drawn += int(idx[-1]) + 1
            last = True
        else:
            drawn += n
            last = False
        lnp = (-np.log(dl[idx] * np.log(dl_hi / dl_lo))
               - 2.0 * np.log(m1[idx]) - np.log(1.0 / m_lo - 1.0 / m_hi)
               - np.log(m1[idx] - m_lo))
        keep["dL"].append(dl[idx]); keep["m1d"].append(m1[idx])
        keep["m2d"].append(m2[idx]); keep["lnp"].append(lnp)
        got += len(idx)
        if last:
            break
    out = {k: np.concatenate(v) if v else np.empty(0) for k, v in keep.items()}
    return out["dL"], out["m1d"], out["m2d"], out["lnp"], drawn


def make_workload(name: str = "tiny", catalog: int = 0, *, n_events=None, n_samples=None,
                  n_grid=None, n_gal=None, n_lambda=None, n_det=None, n_inj_draw=None,
                  seed_offset: int = 0) -> Workload:
    """Build one of BASELINE.json's configs (optionally scaled down by overrides).

    seed = 20250402 + config_index*1000 + catalog_index (+ seed_offset)."""
    cfg = dict(CONFIGS[name])
    for k, v in dict(n_events=n_events, n_samples=n_samples, n_grid=n_grid, n_gal=n_gal,
                     n_lambda=n_lambda, n_det=n_det, n_inj_draw=n_inj_draw).items():
        if v is not None:
            cfg[k] = v
            if k == "n_det":
                cfg["n_inj_draw"] = None
            if k == "n_inj_draw":
                cfg["n_det"] = None
    seed = 20250402 + cfg["index"] * 1000 + catalog + seed_offset
    ss = np.random.SeedSequence(seed).spawn(8)
    r_z, r_m, r_s, r_gal, r_lam, r_inj, r_sm, _ = [np.random.default_rng(s) for s in ss]

    fid = dict(FIDUCIAL)
    if name in ("o5_spec", "o5_photo"):
        fid["Xi0"] = XI0_CATALOGS[catalog]
    fidv = np.array([fid[k] for k in LAMBDA_NAMES])
    ne, ns, nz, ngal = cfg["n_events"], cfg["n_samples"], cfg["n_grid"], cfg["n_gal"]

    cos = _Cosmo(fid["H0"], fid["Om"], fid["Xi0"], fid["n"])
    # events: z_true ~ psi(z) dVc/dz / (1+z) on [0, 1.5]  (eq. 23's integrand)
    zz = np.linspace(1e-4, Z_EVENT_MAX, 20_001)
    pdf_z = _psi(zz, fid["gamma"], fid["kappa"], fid["z_p"]) * np.interp(zz, cos.z, cos.dvdz) / (1 + zz)
    z_true = _inv_cdf_draw(r_z, zz, pdf_z, ne)
    dl_true = cos.dl_of_z(z_true)
    m1s, m2s = _draw_source_masses(r_m, ne, fid)
    m1d_true = m1s * (1 + z_true)
    m2d_true = m2s * (1 + z_true)

    eps = r_s.standard_normal((3, ne, ns))
    dL = dl_true[:, None] * np.exp(0.10 * eps[0])
    a = m1d_true[:, None] * (1 + 0.05 * eps[1])
    b = m2d_true[:, None] * (1 + 0.05 * eps[2])
    m1d = np.maximum(a, b)
    m2d = np.minimum(a, b)
    ln_prior = 2.0 * np.log(dL)

    # lambda batch
    lam = draw_lambda_batch(r_lam, cfg["n_lambda"], fid)

    # redshift grids: extremes of z(dL_true e^{-+0.3}; lambda) over the 16 box corners
    if name == "tiny" and cfg["n_lambda"] == 1:
        corners = [(fid["H0"], fid["Om"], fid["Xi0"], fid["n"])]
    else:
        corners = [(h, o, x, n) for h in LAMBDA_BOX["H0"] for o in LAMBDA_BOX["Om"]
                   for x in LAMBDA_BOX["Xi0"] for n in LAMBDA_BOX["n"]]
    z_lo = np.full(ne, np.inf)
    z_hi = np.zeros(ne)
    for (h, o, x, n) in corners:
        c = _Cosmo(h, o, x, n, n_tab=60_001)
        z_lo = np.minimum(z_lo, c.z_of_dl(dl_true * np.exp(-0.3)))
        z_hi = np.maximum(z_hi, c.z_of_dl(dl_true * np.exp(+0.3)))
    t = np.linspace(0.0, 1.0, nz)
    z_grid = z_lo[:, None] + (z_hi - z_lo)[:, None] * t[None, :]

    # p_gal: N_gal galaxies ~ dVc/dz (fiducial) on the grid range, first one = z_true
    p_gal = np.empty((ne, nz))
    for i in range(ne):
        zf = np.linspace(z_lo[i], z_hi[i], 4001)
        zg = _inv_cdf_draw(r_gal, zf, np.interp(zf, cos.z, cos.dvdz), ngal)
        zg[0] = z_true[i]
        sg = cfg["sigma_z"] * (1 + zg)
        acc = np.zeros(nz)
        for s0 in range(0, ngal, 256):
            d = (z_grid[i][:, None] - zg[None, s0:s0 + 256]) / sg[None, s0:s0 + 256]
            acc += np.sum(np.exp(-0.5 * d * d) / (sg[None, s0:s0 + 256] * np.sqrt(2 * np.pi)), axis=1)
        p_gal[i] = acc / ngal

    inj = draw_injections(r_inj, n_det=cfg.get("n_det"), n_draw=cfg.get("n_inj_draw"))

    return Workload(
        name=name, seed=seed, fiducial=fidv,
        sample_off=np.arange(ne + 1, dtype=np.int64) * ns,
        dL=dL.ravel(), m1d=m1d.ravel(), m2d=m2d.ravel(), ln_prior=ln_prior.ravel(),
        grid_off=np.arange(ne + 1, dtype=np.int64) * nz,
        z_grid=z_grid.ravel(), p_gal=p_gal.ravel(), z_true=z_true, lam=lam,
        inj_dL=inj[0], inj_m1d=inj[1], inj_m2d=inj[2], inj_ln_pdraw=inj[3],
        n_inj_total=int(inj[4]), meta=dict(cfg, catalog=catalog),
    )


def split_into_pixels(w: Workload, n_pix: int = 8, rho: float = 0.4, min_samples: int = 24, same_p_gal: bool = False,
                      seed_offset: int = 0) -> Workload:
    """Stand-in for the paper's sky pixelisation (the sky posteriors are not in the container):
    every event's samples are distributed over n_pix pixels of unequal population, with a sky coordinate correlated
    (coefficient rho) with the sample's distance; each pixel keeps the event's grid and gets its own p_gal (the event's
    one modulated smoothly along z, non-negative); the pixel factor is the fraction of the samples it holds (what a sky
    KDE at the pixel centre times the pixel area estimates).  Returns a workload of sub-events with group_off / ln_factor."""
    rng = np.random.default_rng(np.random.SeedSequence([w.seed, 77, seed_offset]))
    so, dl, m1, m2, lp, go, zg, pg, lnf, goff = [0], [], [], [], [], [0], [], [], [], [0]
    for i in range(w.n_events):
        s = slice(w.sample_off[i], w.sample_off[i + 1])
        g = slice(w.grid_off[i], w.grid_off[i + 1])
        ns = s.stop - s.start
        x = np.log(w.dL[s])
        key = rho * (x - x.mean()) / (x.std() + 1e-300) + np.sqrt(1 - rho * rho) * rng.standard_normal(ns)
        frac = rng.dirichlet(np.full(n_pix, 3.0))
        cnt = np.maximum(min_samples, np.floor(frac * ns).astype(int))
        while cnt.sum() > ns:
            cnt[np.argmax(cnt)] -= 1
        cnt[np.argmax(cnt)] += ns - cnt.sum()
        order = np.argsort(key, kind="stable")
        z = w.z_grid[g]
        start = 0
        for k in range(n_pix):
            idx = np.sort(order[start:start + cnt[k]])          # keep the caller's sample order inside the pixel
            start += cnt[k]
            dl.append(w.dL[s][idx]); m1.append(w.m1d[s][idx]); m2.append(w.m2d[s][idx]); lp.append(w.ln_prior[s][idx])
            so.append(so[-1] + idx.size)
            zg.append(z)
            mod = 1.0 if same_p_gal else 1.0 + 0.6 * np.cos(2 * np.pi * (k / n_pix + 3.0 * (z - z[0]) / (z[-1] - z[0])))
            pg.append(w.p_gal[g] * mod)
            go.append(go[-1] + z.size)
            lnf.append(np.log(idx.size / ns))
        goff.append(goff[-1] + n_pix)
    return dataclasses.replace(
        w, sample_off=np.array(so, dtype=np.int64), dL=np.concatenate(dl), m1d=np.concatenate(m1), m2d=np.concatenate(m2),
        ln_prior=np.concatenate(lp), grid_off=np.array(go, dtype=np.int64), z_grid=np.concatenate(zg),
        p_gal=np.concatenate(pg), group_off=np.array(goff, dtype=np.int64), ln_factor=np.array(lnf),
        meta=dict(w.meta or {}, n_pix=n_pix))


def append_pixels(w: Workload, g: int, pixels) -> Workload:
    """Append (event, pixel) sub-events to physical event g of a many-1d workload (test helper for sparse pixels).
    pixels = [(dL, m1d, m2d, ln_prior, ln_factor), ...]; the new pixels reuse the grid and p_gal of the event's first one."""
    so, go = w.sample_off, w.grid_off
    cut = lambda a, off: [a[off[i]:off[i + 1]] for i in range(len(off) - 1)]
    dl, m1, m2, lp = cut(w.dL, so), cut(w.m1d, so), cut(w.m2d, so), cut(w.ln_prior, so)
    zg, pg = cut(w.z_grid, go), cut(w.p_gal, go)
    lnf = list(w.ln_factor)
    k0, k1 = int(w.group_off[g]), int(w.group_off[g + 1])
    for n, (a, b, c, d, f) in enumerate(pixels):
        for lst, v in ((dl, a), (m1, b), (m2, c), (lp, d), (zg, zg[k0]), (pg, pg[k0])):
            lst.insert(k1 + n, np.asarray(v, dtype=np.float64))
        lnf.insert(k1 + n, float(f))
    goff = w.group_off.copy()
    goff[g + 1:] += len(pixels)
    off = lambda parts: np.concatenate([[0], np.cumsum([len(x) for x in parts])]).astype(np.int64)
    return dataclasses.replace(w, sample_off=off(dl), dL=np.concatenate(dl), m1d=np.concatenate(m1), m2d=np.concatenate(m2),
                               ln_prior=np.concatenate(lp), grid_off=off(zg), z_grid=np.concatenate(zg), p_gal=np.concatenate(pg),
                               group_off=goff, ln_factor=np.array(lnf))
