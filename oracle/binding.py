"""ctypes wrapper around oracle/libchim_oracle.so (argument marshalling only)."""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

PLACE_SAMPLES, PLACE_GRID = 0, 1
BW_SCOTT, BW_FIXED = 0, 1
KERNEL_GAUSS, KERNEL_EPANECHNIKOV = 0, 1
F_LAMBDA_DOMAIN, F_DL_NONMONOTONE, F_EVENT_ZERO, F_XI_ZERO = 1, 2, 4, 8
F_NEFF_LOW, F_TABLE_RANGE, F_BW_DEGENERATE = 16, 32, 64

_lib = None
_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int64)


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
        _lib.chimo_scott_bw.restype = C.c_double
        _lib.chimo_scott_bw_log.restype = C.c_double
        _lib.chimo_event_integral.restype = C.c_double
        _lib.chimo_event_logI.restype = C.c_double
        _lib.chimo_neff.restype = C.c_double
        _lib.chimo_pgal.restype = C.c_double
        _lib.chimo_init()
    return _lib


def _d(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _p(a):
    return None if a is None else a.ctypes.data_as(_dp)


def _lam(lam):
    lam = _d(lam)
    assert lam.shape[-1] == 15
    return lam


def num_threads():
    return int(lib().chimo_num_threads())


def distances(lam, z):
    lam, z = _lam(lam), _d(np.atleast_1d(z))
    out = [np.empty_like(z) for _ in range(4)]
    lib().chimo_distances(_p(lam), C.c_int(z.size), _p(z), *[_p(o) for o in out])
    return dict(dc=out[0], dl_em=out[1], dl_gw=out[2], ddl_gw_dz=out[3])


def volume(lam, z):
    lam, z = _lam(lam), _d(np.atleast_1d(z))
    dv, vc = np.empty_like(z), np.empty_like(z)
    lib().chimo_volume(_p(lam), C.c_int(z.size), _p(z), _p(dv), _p(vc))
    return dv, vc


def dl_monotone(lam, z_table_max=10.0, n_table=2048):
    return bool(lib().chimo_dl_monotone(_p(_lam(lam)), C.c_double(z_table_max), C.c_int(n_table)))


def z_of_dl(lam, dl, z_table_max=10.0):
    lam, dl = _lam(lam), _d(np.atleast_1d(dl))
    z = np.empty_like(dl)
    lib().chimo_z_of_dl(_p(lam), C.c_double(z_table_max), C.c_int(dl.size), _p(dl), _p(z))
    return z


def smoothing(lam, m):
    lam, m = _lam(lam), _d(np.atleast_1d(m))
    o = np.empty_like(m)
    lib().chimo_smoothing(_p(lam), C.c_int(m.size), _p(m), _p(o))
    return o


def p_m1(lam, m):
    lam, m = _lam(lam), _d(np.atleast_1d(m))
    o = np.empty_like(m)
    lib().chimo_p_m1(_p(lam), C.c_int(m.size), _p(m), _p(o))
    return o


def p_m2_given_m1(lam, m1, m2):
    lam, m1, m2 = _lam(lam), _d(np.atleast_1d(m1)), _d(np.atleast_1d(m2))
    o = np.empty_like(m1)
    lib().chimo_p_m2_given_m1(_p(lam), C.c_int(m1.size), _p(m1), _p(m2), _p(o))
    return o


def mass_pdf(lam, m1, m2):
    lam, m1, m2 = _lam(lam), _d(np.atleast_1d(m1)), _d(np.atleast_1d(m2))
    o = np.empty_like(m1)
    lib().chimo_mass_pdf(_p(lam), C.c_int(m1.size), _p(m1), _p(m2), _p(o))
    return o


def ln_smoothing(lam, m):
    lam, m = _lam(lam), _d(np.atleast_1d(m))
    o = np.empty_like(m)
    lib().chimo_ln_smoothing(_p(lam), C.c_int(m.size), _p(m), _p(o))
    return o


def ln_p_m2_given_m1(lam, m1, m2):
    lam, m1, m2 = _lam(lam), _d(np.atleast_1d(m1)), _d(np.atleast_1d(m2))
    o = np.empty_like(m1)
    lib().chimo_ln_p_m2_given_m1(_p(lam), C.c_int(m1.size), _p(m1), _p(m2), _p(o))
    return o


def ln_mass_pdf(lam, m1, m2):
    lam, m1, m2 = _lam(lam), _d(np.atleast_1d(m1)), _d(np.atleast_1d(m2))
    o = np.empty_like(m1)
    lib().chimo_ln_mass_pdf(_p(lam), C.c_int(m1.size), _p(m1), _p(m2), _p(o))
    return o


def psi(lam, z):
    lam, z = _lam(lam), _d(np.atleast_1d(z))
    o = np.empty_like(z)
    lib().chimo_psi(_p(lam), C.c_int(z.size), _p(z), _p(o))
    return o


def sample_weights(lam, dl, m1d, m2d, ln_prior, placement=PLACE_SAMPLES, z_table_max=10.0):
    lam, dl, m1d, m2d, lp = _lam(lam), _d(dl), _d(m1d), _d(m2d), _d(ln_prior)
    z, w = np.empty_like(dl), np.empty_like(dl)
    rf = C.c_int(0)
    lib().chimo_sample_weights(_p(lam), C.c_int(placement), C.c_double(z_table_max), C.c_int(dl.size),
                               _p(dl), _p(m1d), _p(m2d), _p(lp), _p(z), _p(w), C.byref(rf))
    return z, w, bool(rf.value)


def sample_log_weights(lam, dl, m1d, m2d, ln_prior, placement=PLACE_SAMPLES, z_table_max=10.0):
    """O6 in log space: (z_j, ln w_j, range flag); ln w = -inf where the weight is 0."""
    lam, dl, m1d, m2d, lp = _lam(lam), _d(dl), _d(m1d), _d(m2d), _d(ln_prior)
    z, lw = np.empty_like(dl), np.empty_like(dl)
    rf = C.c_int(0)
    lib().chimo_sample_log_weights(_p(lam), C.c_int(placement), C.c_double(z_table_max), C.c_int(dl.size),
                                   _p(dl), _p(m1d), _p(m2d), _p(lp), _p(z), _p(lw), C.byref(rf))
    return z, lw, bool(rf.value)


def scott_bw_log(z, lw):
    """O7 from log weights (the form the event path uses)."""
    z, lw = _d(z), _d(lw)
    return float(lib().chimo_scott_bw_log(C.c_int(z.size), _p(z), _p(lw)))


def scott_bw(z, w):
    z, w = _d(z), _d(w)
    return float(lib().chimo_scott_bw(C.c_int(z.size), _p(z), _p(w)))


def kde(z, w, h, zg):
    z, w, zg = _d(z), _d(w), _d(zg)
    K = np.empty_like(zg)
    lib().chimo_kde(C.c_int(z.size), _p(z), _p(w), C.c_double(h), C.c_int(zg.size), _p(zg), _p(K))
    return K


def kde_epanechnikov(z, w, h, zg):
    """O8': Epanechnikov kernel with the same standard deviation h as the Gaussian one (h_E = sqrt(5) h, reading R19)."""
    z, w, zg = _d(z), _d(w), _d(zg)
    K = np.empty_like(zg)
    lib().chimo_kde_epan(C.c_int(z.size), _p(z), _p(w), C.c_double(h), C.c_int(zg.size), _p(zg), _p(K))
    return K


def bin_samples(z, w, n_bins):
    """R23: equal-width bins on [min z, max z]; pseudo-samples (weighted mean z, sum of weights)."""
    z, w = _d(z), _d(w)
    zb, wb = np.empty(n_bins), np.empty(n_bins)
    n = lib().chimo_bin_samples(C.c_int(z.size), _p(z), _p(w), C.c_int(n_bins), _p(zb), _p(wb))
    return zb[:n], wb[:n]


def event_integral(lam, zg, K, pgal, placement=PLACE_SAMPLES):
    lam, zg, K, pgal = _lam(lam), _d(zg), _d(K), _d(pgal)
    return float(lib().chimo_event_integral(_p(lam), C.c_int(placement), C.c_int(zg.size), _p(zg), _p(K), _p(pgal)))


def event_logI(lam, dl, m1d, m2d, ln_prior, zg, pgal, placement=PLACE_SAMPLES, bw_rule=BW_SCOTT,
               fixed_bw=float("nan"), z_table_max=10.0, kernel=KERNEL_GAUSS, n_bins=0):
    lib().chimo_set_kernel(C.c_int(kernel))
    lib().chimo_set_bins(C.c_int(n_bins))
    lam, dl, m1d, m2d, lp, zg, pgal = _lam(lam), _d(dl), _d(m1d), _d(m2d), _d(ln_prior), _d(zg), _d(pgal)
    h = C.c_double(0.0)
    fl = C.c_uint32(0)
    v = lib().chimo_event_logI(_p(lam), C.c_int(placement), C.c_int(bw_rule), C.c_double(fixed_bw),
                               C.c_double(z_table_max), C.c_int(dl.size), _p(dl), _p(m1d), _p(m2d), _p(lp),
                               C.c_int(zg.size), _p(zg), _p(pgal), C.byref(h), C.byref(fl))
    return float(v), float(h.value), int(fl.value)


def pcat(lam, z_gal, sigma_gal, zg, w_gal=None):
    """PAPER.md:62 eq. 8 for one line of sight: catalogue redshift density on the grid zg (reading R22)."""
    lam, zt, st, zg = _lam(lam), _d(z_gal), _d(sigma_gal), _d(zg)
    wg = None if w_gal is None else _d(w_gal)
    out = np.empty_like(zg)
    lib().chimo_pcat(_p(lam), C.c_int(zt.size), _p(zt), _p(st), _p(wg), C.c_int(zg.size), _p(zg), _p(out))
    return out


def pgal(lam, z_max, z_gal, sigma_gal, z_compl, p_compl, zg, w_gal=None):
    """PAPER.md:58 eq. 7 with eq. 9-10 for one line of sight (reading R25): returns (p_gal on zg, f_R)."""
    lam, zt, st, zc, pc, zg = _lam(lam), _d(z_gal), _d(sigma_gal), _d(z_compl), _d(p_compl), _d(zg)
    wg = None if w_gal is None else _d(w_gal)
    out = np.empty_like(zg)
    fr = lib().chimo_pgal(_p(lam), C.c_double(z_max), C.c_int(zt.size), _p(zt), _p(st), _p(wg), C.c_int(zc.size), _p(zc), _p(pc),
                          C.c_int(zg.size), _p(zg), _p(out))
    return out, float(fr)


def selection_sums(lam, dl, m1d, m2d, ln_pdraw, z_cat_max=1.5, z_table_max=10.0, return_s=False):
    lam, dl, m1d, m2d, lp = _lam(lam), _d(dl), _d(m1d), _d(m2d), _d(ln_pdraw)
    s1, s2 = C.c_double(0), C.c_double(0)
    rf = C.c_int(0)
    s = np.empty_like(dl) if return_s else None
    lib().chimo_selection_sums(_p(lam), C.c_double(z_cat_max), C.c_double(z_table_max), C.c_int64(dl.size),
                               _p(dl), _p(m1d), _p(m2d), _p(lp), C.byref(s1), C.byref(s2), _p(s), C.byref(rf))
    if return_s:
        return s1.value, s2.value, s
    return s1.value, s2.value


def neff(sum_s, sum_s2, n_inj_total):
    return float(lib().chimo_neff(C.c_double(sum_s), C.c_double(sum_s2), C.c_double(n_inj_total)))


def loglike_batch(lam, sample_off, dl, m1d, m2d, ln_prior, grid_off, zg, pgal, *, fixed_bw=None,
                  inj=None, n_inj_total=0, placement=PLACE_SAMPLES, bw_rule=BW_SCOTT, z_cat_max=1.5,
                  z_table_max=10.0, n_table=2048, neff_factor=5.0, kernel=KERNEL_GAUSS, group_off=None, ln_factor=None, n_bins=0):
    """inj = (dL, m1d, m2d, ln_pdraw) of the detected set or None.  Returns a dict of arrays."""
    lib().chimo_set_kernel(C.c_int(kernel))
    lib().chimo_set_bins(C.c_int(n_bins))
    lam = np.atleast_2d(_lam(lam))
    nl = lam.shape[0]
    so = np.ascontiguousarray(sample_off, dtype=np.int64)
    go = np.ascontiguousarray(grid_off, dtype=np.int64)
    ne = so.size - 1
    dl, m1d, m2d, lp, zg, pgal = map(_d, (dl, m1d, m2d, ln_prior, zg, pgal))
    fb = None if fixed_bw is None else _d(fixed_bw)
    if inj is None:
        nd, i0, i1, i2, i3 = 0, None, None, None, None
    else:
        i0, i1, i2, i3 = map(_d, inj)
        nd = i0.size
    out = dict(loglike=np.empty(nl), event_logI=np.empty((nl, ne)), logxi=np.empty(nl), neff=np.empty(nl),
               h=np.empty((nl, ne)), flags=np.zeros(nl, dtype=np.uint32))
    if group_off is not None:
        gof = np.ascontiguousarray(group_off, dtype=np.int64)
        lnf = _d(ln_factor)
        assert gof[0] == 0 and gof[-1] == ne and lnf.size == ne
        ng, gp, fp = gof.size - 1, gof.ctypes.data_as(_ip), _p(lnf)
    else:
        ng, gp, fp = 0, None, None
    lib().chimo_loglike_batch_grouped(
        C.c_int(nl), _p(lam), C.c_int(placement), C.c_int(bw_rule), C.c_double(z_cat_max),
        C.c_double(z_table_max), C.c_int(n_table), C.c_double(neff_factor), C.c_int(ne),
        so.ctypes.data_as(_ip), _p(dl), _p(m1d), _p(m2d), _p(lp), go.ctypes.data_as(_ip), _p(zg), _p(pgal),
        _p(fb), C.c_int64(nd), C.c_double(float(n_inj_total)), _p(i0), _p(i1), _p(i2), _p(i3),
        C.c_int(ng), gp, fp,
        _p(out["loglike"]), _p(out["event_logI"]), _p(out["logxi"]), _p(out["neff"]), _p(out["h"]),
        out["flags"].ctypes.data_as(C.POINTER(C.c_uint32)))
    return out


def loglike_workload(w, lam=None, **kw):
    """Convenience: run the oracle on a workloads.Workload."""
    lam = w.lam if lam is None else lam
    inj = (w.inj_dL, w.inj_m1d, w.inj_m2d, w.inj_ln_pdraw) if w.n_det > 0 else None
    kw.setdefault("z_cat_max", w.z_cat_max)
    if getattr(w, "group_off", None) is not None:
        kw.setdefault("group_off", w.group_off)
        kw.setdefault("ln_factor", w.ln_factor)
    return loglike_batch(lam, w.sample_off, w.dL, w.m1d, w.m2d, w.ln_prior, w.grid_off, w.z_grid, w.p_gal,
                         inj=inj, n_inj_total=w.n_inj_total, **kw)


def loglike_grad(w, lam, rel_step=1e-2, **kw):
    """Gradient of log L with respect to the 15 hyper-parameters at ONE lambda, by its definition as a limit of difference
    quotients: central differences of the fp64 oracle with one Richardson step,
        g_k = [4 D(h_k / 2) - D(h_k)] / 3,  D(h) = [logL(lam + h e_k) - logL(lam - h e_k)] / 2h,  h_k = rel_step |lam_k| (rel_step if 0).
    Returns (logL(lam), g[15])."""
    lam = _lam(lam).reshape(15)
    rows = [lam]
    hs = []
    for k in range(15):
        h = rel_step * abs(lam[k]) if lam[k] != 0.0 else rel_step
        hs.append(h)
        for d in (1.0, -1.0, 0.5, -0.5):
            r = lam.copy()
            r[k] += d * h
            rows.append(r)
    f = loglike_workload(w, lam=np.array(rows), **kw)["loglike"]
    g = np.empty(15)
    for k in range(15):
        d1 = (f[1 + 4 * k] - f[2 + 4 * k]) / (2.0 * hs[k])
        d2 = (f[3 + 4 * k] - f[4 + 4 * k]) / hs[k]
        g[k] = (4.0 * d2 - d1) / 3.0
    return float(f[0]), g
