"""ctypes binding of libchim.so: same names as include/chim.h, plus a small Context convenience class."""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))

CHIM_MEM_HOST, CHIM_MEM_DEVICE = 0, 1
CHIM_ON_SAMPLES, CHIM_ON_GRID = 0, 1
CHIM_BW_SCOTT, CHIM_BW_FIXED = 0, 1
CHIM_KDE_AUTO, CHIM_KDE_DIRECT, CHIM_KDE_POWER, CHIM_KDE_NONE = 0, 1, 2, 3
CHIM_KERNEL_GAUSS, CHIM_KERNEL_EPANECHNIKOV = 0, 1
CHIM_FLAG_LAMBDA_DOMAIN, CHIM_FLAG_DL_NONMONOTONE, CHIM_FLAG_EVENT_ZERO, CHIM_FLAG_XI_ZERO = 1, 2, 4, 8
CHIM_FLAG_NEFF_LOW, CHIM_FLAG_TABLE_RANGE, CHIM_FLAG_BW_DEGENERATE = 16, 32, 64
CHIM_PCAT_STATIC_MAX_GALAXIES = 262144
N_LAMBDA_PARAMS = 15


class ChimError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__(f"libchim status {status}: {msg}")
        self.status = status


class ChimConfig(C.Structure):
    _fields_ = [("device", C.c_int32), ("mem", C.c_int32), ("stream", C.c_void_p), ("placement", C.c_int32),
                ("bw_rule", C.c_int32), ("kde_cutoff", C.c_double), ("z_cat_max", C.c_double),
                ("z_table_max", C.c_double), ("n_table", C.c_int32), ("n_dl_table", C.c_int32),
                ("n_win_table", C.c_int32), ("lambda_chunk", C.c_int32), ("neff_factor", C.c_double),
                ("kde_method", C.c_int32), ("n_mass_table", C.c_int32), ("count_pairs", C.c_int32),
                ("kde_kernel", C.c_int32), ("n_bins", C.c_int32)]


class ChimStats(C.Structure):
    _fields_ = [("kde_pairs_evaluated", C.c_uint64), ("kde_pairs_in_cutoff", C.c_uint64), ("kde_pairs_dense", C.c_uint64), ("sample_evals", C.c_uint64),
                ("injection_evals", C.c_uint64), ("kernel_launches", C.c_uint64)]


class ChimKernelTimes(C.Structure):
    _fields_ = [("tables_ms", C.c_double), ("events_ms", C.c_double), ("inject_ms", C.c_double),
                ("combine_ms", C.c_double), ("tables_launches", C.c_uint32), ("events_launches", C.c_uint32),
                ("inject_launches", C.c_uint32), ("combine_launches", C.c_uint32), ("events_general_ms", C.c_double),
                ("events_general_launches", C.c_uint32), ("events_handed_over", C.c_uint32)]


class ChimAluPeaks(C.Structure):
    _fields_ = [("ex2_gops", C.c_double), ("ffma_gops", C.c_double), ("dfma_gops", C.c_double),
                ("ffma2_gops", C.c_double), ("sm_count", C.c_int32), ("reserved", C.c_int32)]


_lib = None
_vp, _dp, _ip, _up = C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p   # raw addresses (host or device)


def lib_path() -> str:
    return os.path.join(HERE, "libchim.so")


def lib():
    """Load libchim.so (fails loudly if it is missing: there is no fallback path)."""
    global _lib
    if _lib is not None:
        return _lib
    p = lib_path()
    if not os.path.exists(p):
        raise ImportError(f"{p} not found: build it with `python -m paper_2504_02034_b200.build` "
                          "(nvcc, sm_100a). There is no CPU or PyTorch fallback.")
    L = C.CDLL(p)
    L.chim_build_id.restype = C.c_char_p
    from . import build as _build
    have, want = L.chim_build_id().decode(), _build.source_hash()
    if have != want:
        raise ImportError(f"{p} was built from other sources (build id {have}, sources {want}): rebuild it with "
                          "`python -m paper_2504_02034_b200.build`. A stale library is never used.")
    L.chim_default_config.argtypes = [C.POINTER(ChimConfig)]
    L.chim_default_config.restype = None
    L.chim_create.argtypes = [C.POINTER(ChimConfig), C.POINTER(C.c_void_p)]
    L.chim_destroy.argtypes = [C.c_void_p]
    L.chim_destroy.restype = None
    L.chim_last_error.argtypes = [C.c_void_p]
    L.chim_last_error.restype = C.c_char_p
    L.chim_version.restype = C.c_int
    L.chim_init_events.argtypes = [C.c_void_p, C.c_int32] + [C.c_void_p] * 9
    L.chim_init_injections.argtypes = [C.c_void_p, C.c_int64, C.c_int64] + [C.c_void_p] * 4
    L.chim_set_event_groups.argtypes = [C.c_void_p, C.c_int32, C.c_void_p, C.c_void_p]
    L.chim_build_pcat.argtypes = [C.c_void_p, C.c_double, C.c_int32] + [C.c_void_p] * 7
    L.chim_build_pgal.argtypes = [C.c_void_p, C.c_double, C.c_double, C.c_int32] + [C.c_void_p] * 11
    L.chim_build_pcat_static.argtypes = [C.c_void_p, C.c_double, C.c_int32, C.c_int64] + [C.c_void_p] * 7
    L.chim_loglike_batch.argtypes = [C.c_void_p, C.c_int32] + [C.c_void_p] * 6
    L.chim_loglike_batch_host.argtypes = [C.c_void_p, C.c_int32] + [C.c_void_p] * 6
    L.chim_loglike_grad_batch.argtypes = [C.c_void_p, C.c_int32, C.c_void_p, C.c_double, C.c_void_p, C.c_void_p, C.c_void_p]
    L.chim_get_stats.argtypes = [C.c_void_p, C.POINTER(ChimStats)]
    L.chim_set_profiling.argtypes = [C.c_void_p, C.c_int32]
    L.chim_get_kernel_times.argtypes = [C.c_void_p, C.POINTER(ChimKernelTimes)]
    L.chim_measure_alu_peaks.argtypes = [C.c_void_p, C.POINTER(ChimAluPeaks)]
    L.chim_debug_table_lookup.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p]
    L.chim_debug_event_samples.argtypes = [C.c_void_p, C.c_void_p, C.c_int32, C.c_void_p, C.c_void_p]
    L.chim_debug_event_kde.argtypes = [C.c_void_p, C.c_void_p, C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p]
    L.chim_debug_injection_weights.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
    _lib = L
    return L


# ---- same-name wrappers (status -> exception) ---------------------------------------------------------
def _check(ctx, status):
    if status != 0:
        msg = lib().chim_last_error(ctx).decode() if ctx else "no context"
        raise ChimError(status, msg)


def _addr(a):
    """Address of a numpy array (host) or torch tensor (device or host); None -> NULL."""
    if a is None:
        return None
    if isinstance(a, np.ndarray):
        assert a.flags["C_CONTIGUOUS"]
        return a.ctypes.data
    return a.data_ptr()


def chim_version():
    return int(lib().chim_version())


def chim_default_config() -> ChimConfig:
    cfg = ChimConfig()
    lib().chim_default_config(C.byref(cfg))
    return cfg


def chim_create(cfg: ChimConfig | None = None):
    h = C.c_void_p()
    st = lib().chim_create(C.byref(cfg) if cfg is not None else None, C.byref(h))
    if st != 0:
        raise ChimError(st, lib().chim_last_error(None).decode() or "chim_create failed")
    return h


def chim_destroy(ctx):
    lib().chim_destroy(ctx)


def chim_last_error(ctx) -> str:
    return lib().chim_last_error(ctx).decode()


def chim_init_events(ctx, n_events, sample_off, dL, m1d, m2d, ln_prior, grid_off, z_grid, p_gal, fixed_bw=None):
    _check(ctx, lib().chim_init_events(ctx, n_events, *[_addr(a) for a in (sample_off, dL, m1d, m2d, ln_prior,
                                                                           grid_off, z_grid, p_gal, fixed_bw)]))


def chim_set_event_groups(ctx, n_groups, group_off, ln_factor):
    _check(ctx, lib().chim_set_event_groups(ctx, n_groups, _addr(group_off), _addr(ln_factor)))


def chim_build_pcat(ctx, omega_m, n_los, gal_off, z_gal, sigma_gal, w_gal, grid_off, z_grid, p_cat_out):
    _check(ctx, lib().chim_build_pcat(ctx, omega_m, n_los, *[_addr(a) for a in (gal_off, z_gal, sigma_gal, w_gal, grid_off,
                                                                               z_grid, p_cat_out)]))


def chim_build_pcat_static(ctx, omega_m, n_los, n_gal_total, gal_off, z_gal, sigma_gal, w_gal, grid_off, z_grid, p_cat_out):
    """chim_build_pcat for callers that must not allocate device memory (include/chim.h): DEVICE pointers only, enqueue-only."""
    _check(ctx, lib().chim_build_pcat_static(ctx, omega_m, n_los, n_gal_total, *[_addr(a) for a in (gal_off, z_gal, sigma_gal, w_gal,
                                                                                                  grid_off, z_grid, p_cat_out)]))


def chim_build_pgal(ctx, omega_m, z_max, n_los, gal_off, z_gal, sigma_gal, w_gal, compl_off, z_compl, p_compl, grid_off, z_grid,
                    p_gal_out, f_r_out=None):
    _check(ctx, lib().chim_build_pgal(ctx, omega_m, z_max, n_los, *[_addr(a) for a in (gal_off, z_gal, sigma_gal, w_gal, compl_off,
                                                                                       z_compl, p_compl, grid_off, z_grid, p_gal_out,
                                                                                       f_r_out)]))


def chim_init_injections(ctx, n_det, n_inj_total, dL, m1d, m2d, ln_pdraw):
    _check(ctx, lib().chim_init_injections(ctx, n_det, n_inj_total, *[_addr(a) for a in (dL, m1d, m2d, ln_pdraw)]))


def chim_loglike_batch(ctx, n_lambda, lam, out_loglike, out_event_logI=None, out_logxi=None, out_neff=None,
                       out_flags=None):
    _check(ctx, lib().chim_loglike_batch(ctx, n_lambda, *[_addr(a) for a in (lam, out_loglike, out_event_logI,
                                                                              out_logxi, out_neff, out_flags)]))


def chim_loglike_batch_host(ctx, n_lambda, lam, out_loglike, out_event_logI=None, out_logxi=None, out_neff=None,
                            out_flags=None):
    _check(ctx, lib().chim_loglike_batch_host(ctx, n_lambda, *[_addr(a) for a in (lam, out_loglike, out_event_logI,
                                                                                   out_logxi, out_neff, out_flags)]))


def chim_loglike_grad_batch(ctx, n_lambda, lam, rel_step, out_loglike, out_grad, out_flags=None):
    _check(ctx, lib().chim_loglike_grad_batch(ctx, n_lambda, _addr(lam), rel_step, _addr(out_loglike), _addr(out_grad), _addr(out_flags)))


def chim_get_stats(ctx) -> ChimStats:
    s = ChimStats()
    _check(ctx, lib().chim_get_stats(ctx, C.byref(s)))
    return s


def chim_measure_alu_peaks(ctx) -> ChimAluPeaks:
    p = ChimAluPeaks()
    _check(ctx, lib().chim_measure_alu_peaks(ctx, C.byref(p)))
    return p


# ---- convenience ------------------------------------------------------------------------------------
def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


class Context:
    """One libchim context bound to a CUDA device and stream (torch supplies both)."""

    def __init__(self, device=0, stream=None, placement=CHIM_ON_SAMPLES, bw_rule=CHIM_BW_SCOTT, kde_cutoff=None,
                 z_cat_max=None, z_table_max=None, n_table=None, n_dl_table=None, n_win_table=None,
                 lambda_chunk=None, neff_factor=None, kde_method=None, n_mass_table=None, count_pairs=None,
                 kde_kernel=None, n_bins=None):
        import torch
        if not torch.cuda.is_available():
            raise ChimError(-3, "no CUDA device: libchim has no CPU fallback")
        self.torch = torch
        self.device = torch.device("cuda", device)
        cfg = chim_default_config()
        cfg.device = device
        cfg.mem = CHIM_MEM_HOST
        if stream is None:
            stream = torch.cuda.current_stream(self.device)
        self.stream = stream
        cfg.stream = stream.cuda_stream
        cfg.placement, cfg.bw_rule = placement, bw_rule
        for k, v in dict(kde_cutoff=kde_cutoff, z_cat_max=z_cat_max, z_table_max=z_table_max, n_table=n_table,
                         n_dl_table=n_dl_table, n_win_table=n_win_table, lambda_chunk=lambda_chunk,
                         neff_factor=neff_factor, kde_method=kde_method, n_mass_table=n_mass_table,
                         count_pairs=count_pairs, kde_kernel=kde_kernel, n_bins=n_bins).items():
            if v is not None:
                setattr(cfg, k, v)
        self.cfg = cfg
        self.h = chim_create(cfg)
        self.n_events = 0
        self.n_det = 0
        self._ns = self._nz = None

    def close(self):
        if getattr(self, "h", None):
            chim_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- init ------------------------------------------------------------------------------------------
    def init_events(self, sample_off, dL, m1d, m2d, ln_prior, grid_off, z_grid, p_gal, fixed_bw=None):
        so = np.ascontiguousarray(sample_off, dtype=np.int64)
        go = np.ascontiguousarray(grid_off, dtype=np.int64)
        arrs = [_f64(a) for a in (dL, m1d, m2d, ln_prior)]
        zg, pg = _f64(z_grid), _f64(p_gal)
        fb = None if fixed_bw is None else _f64(fixed_bw)
        chim_init_events(self.h, len(so) - 1, so, *arrs, go, zg, pg, fb)
        self.n_events = len(so) - 1
        self._ns, self._nz = np.diff(so), np.diff(go)

    def build_pcat(self, omega_m, gal_off, z_gal, sigma_gal, grid_off, z_grid, w_gal=None):
        """PAPER.md:62 eq. 8 on the given grids (host arrays in, host array out)."""
        go = np.ascontiguousarray(gal_off, dtype=np.int64)
        po = np.ascontiguousarray(grid_off, dtype=np.int64)
        zg = _f64(z_grid)
        out = np.empty_like(zg)
        chim_build_pcat(self.h, float(omega_m), len(go) - 1, go, _f64(z_gal), _f64(sigma_gal),
                        None if w_gal is None else _f64(w_gal), po, zg, out)
        return out

    def build_pcat_static(self, omega_m, n_gal_total, gal_off, z_gal, sigma_gal, grid_off, z_grid, p_cat_out, w_gal=None):
        """PAPER.md:62 eq. 8 for a caller that cannot let this library allocate on the GPU (the memory belongs to a framework's
        pool, or a cudaMalloc / cudaFree would stall a running batch).  Every array is a CUDA tensor the caller owns -- int64
        offsets, float64 values, p_cat_out included -- and n_gal_total = gal_off[-1] is passed by value (the offsets stay on the
        device).  At most CHIM_PCAT_STATIC_MAX_GALAXIES galaxies per call: the per-galaxy scratch is a fixed array inside
        libchim.so, shared by all calls on the GPU, so calls that may overlap there must not be issued.  Enqueues on the
        context's stream and returns p_cat_out; nothing is validated beyond the sizes."""
        t = self.torch
        for a, dt in ((gal_off, t.int64), (grid_off, t.int64), (z_gal, t.float64), (sigma_gal, t.float64), (z_grid, t.float64),
                      (p_cat_out, t.float64)) + (((w_gal, t.float64),) if w_gal is not None else ()):
            assert a.is_cuda and a.dtype == dt and a.is_contiguous()
        assert p_cat_out.numel() == z_grid.numel() and gal_off.numel() == grid_off.numel()
        chim_build_pcat_static(self.h, float(omega_m), gal_off.numel() - 1, int(n_gal_total), gal_off, z_gal, sigma_gal, w_gal,
                               grid_off, z_grid, p_cat_out)
        return p_cat_out

    def build_pgal(self, omega_m, z_max, gal_off, z_gal, sigma_gal, compl_off, z_compl, p_compl, grid_off, z_grid, w_gal=None):
        """PAPER.md:58 eq. 7 with eq. 9-10 on the given grids (host arrays in); returns (p_gal, f_R per line of sight)."""
        go = np.ascontiguousarray(gal_off, dtype=np.int64)
        co = np.ascontiguousarray(compl_off, dtype=np.int64)
        po = np.ascontiguousarray(grid_off, dtype=np.int64)
        zg = _f64(z_grid)
        out, fr = np.empty_like(zg), np.empty(len(go) - 1)
        chim_build_pgal(self.h, float(omega_m), float(z_max), len(go) - 1, go, _f64(z_gal), _f64(sigma_gal),
                        None if w_gal is None else _f64(w_gal), co, _f64(z_compl), _f64(p_compl), po, zg, out, fr)
        return out, fr

    def set_event_groups(self, group_off, ln_factor):
        """many-1d: the loaded entries are (event, pixel) sub-events; None removes the grouping."""
        if group_off is None:
            chim_set_event_groups(self.h, 0, None, None)
            return
        go = np.ascontiguousarray(group_off, dtype=np.int64)
        chim_set_event_groups(self.h, len(go) - 1, go, _f64(ln_factor))

    def init_injections(self, dL, m1d, m2d, ln_pdraw, n_inj_total):
        arrs = [_f64(a) for a in (dL, m1d, m2d, ln_pdraw)]
        chim_init_injections(self.h, arrs[0].size, int(n_inj_total), *arrs)
        self.n_det = arrs[0].size

    def init_workload(self, w, fixed_bw=None):
        self.init_events(w.sample_off, w.dL, w.m1d, w.m2d, w.ln_prior, w.grid_off, w.z_grid, w.p_gal, fixed_bw)
        if getattr(w, "group_off", None) is not None:
            self.set_event_groups(w.group_off, w.ln_factor)
        if w.n_det > 0:
            self.init_injections(w.inj_dL, w.inj_m1d, w.inj_m2d, w.inj_ln_pdraw, w.n_inj_total)

    # -- hot path --------------------------------------------------------------------------------------
    def alloc_outputs(self, n_lambda, event_logI=True):
        t = self.torch
        o = dict(loglike=t.empty(n_lambda, dtype=t.float64, device=self.device),
                 logxi=t.empty(n_lambda, dtype=t.float64, device=self.device),
                 neff=t.empty(n_lambda, dtype=t.float64, device=self.device),
                 flags=t.empty(n_lambda, dtype=t.int32, device=self.device))
        if event_logI:
            o["event_logI"] = t.empty((n_lambda, self.n_events), dtype=t.float64, device=self.device)
        return o

    def loglike_batch(self, lam, out=None, event_logI=True):
        """lam: torch CUDA float64 [n_lambda, 15].  Enqueues on the context's stream; returns device tensors."""
        t = self.torch
        assert lam.is_cuda and lam.dtype == t.float64 and lam.is_contiguous() and lam.shape[-1] == N_LAMBDA_PARAMS
        n = lam.shape[0]
        if out is None:
            out = self.alloc_outputs(n, event_logI)
        chim_loglike_batch(self.h, n, lam, out["loglike"], out.get("event_logI"), out["logxi"], out["neff"], out["flags"])
        return out

    def loglike_batch_host(self, lam, out=None, event_logI=False):
        """lam: host array [n_lambda, 15] (numpy or pinned torch).  Copies in, computes, copies out, synchronises."""
        n = lam.shape[0]
        if out is None:
            out = dict(loglike=np.empty(n), logxi=np.empty(n), neff=np.empty(n), flags=np.zeros(n, dtype=np.uint32))
            if event_logI:
                out["event_logI"] = np.empty((n, self.n_events))
        chim_loglike_batch_host(self.h, n, lam, out["loglike"], out.get("event_logI"), out["logxi"], out["neff"], out["flags"])
        return out

    def loglike_grad_batch(self, lam, rel_step=1e-2):
        """lam: torch CUDA float64 [n_lambda, 15] -> dict(loglike [n], grad [n, 15], flags [n]) of device tensors."""
        t = self.torch
        assert lam.is_cuda and lam.dtype == t.float64 and lam.is_contiguous() and lam.shape[-1] == N_LAMBDA_PARAMS
        n = lam.shape[0]
        out = dict(loglike=t.empty(n, dtype=t.float64, device=self.device), grad=t.empty((n, N_LAMBDA_PARAMS), dtype=t.float64, device=self.device),
                   flags=t.empty(n, dtype=t.int32, device=self.device))
        chim_loglike_grad_batch(self.h, n, lam, float(rel_step), out["loglike"], out["grad"], out["flags"])
        return out

    def stats(self):
        s = chim_get_stats(self.h)
        return {k: int(getattr(s, k)) for k, _ in ChimStats._fields_}

    def set_profiling(self, on=True):
        _check(self.h, lib().chim_set_profiling(self.h, 1 if on else 0))

    def kernel_times(self):
        k = ChimKernelTimes()
        _check(self.h, lib().chim_get_kernel_times(self.h, C.byref(k)))
        return {n: getattr(k, n) for n, _ in ChimKernelTimes._fields_}

    def alu_peaks(self):
        p = chim_measure_alu_peaks(self.h)
        return {n: getattr(p, n) for n, _ in ChimAluPeaks._fields_ if n != "reserved"}

    # -- diagnostics -----------------------------------------------------------------------------------
    def _lam1(self, lam):
        t = self.torch
        return t.as_tensor(np.asarray(lam, dtype=np.float64).reshape(N_LAMBDA_PARAMS), device=self.device).contiguous()

    def debug_table_lookup(self, lam, dL):
        t = self.torch
        d = t.as_tensor(_f64(dL), device=self.device)
        z, r = t.empty_like(d), t.empty_like(d)
        _check(self.h, lib().chim_debug_table_lookup(self.h, self._lam1(lam).data_ptr(), d.numel(), d.data_ptr(),
                                                     z.data_ptr(), r.data_ptr()))
        return z.cpu().numpy(), r.cpu().numpy()

    def debug_event_samples(self, lam, event):
        t = self.torch
        ns = int(self._ns[event])
        z = t.empty(ns, dtype=t.float64, device=self.device)
        w = t.empty_like(z)
        _check(self.h, lib().chim_debug_event_samples(self.h, self._lam1(lam).data_ptr(), event, z.data_ptr(), w.data_ptr()))
        return z.cpu().numpy(), w.cpu().numpy()

    def debug_event_kde(self, lam, event):
        t = self.torch
        K = t.empty(int(self._nz[event]), dtype=t.float64, device=self.device)
        hl = t.empty(2, dtype=t.float64, device=self.device)
        _check(self.h, lib().chim_debug_event_kde(self.h, self._lam1(lam).data_ptr(), event, hl.data_ptr(), K.data_ptr(),
                                                  hl.data_ptr() + 8))
        hl = hl.cpu().numpy()
        return float(hl[0]), K.cpu().numpy(), float(hl[1])

    def debug_injection_weights(self, lam):
        t = self.torch
        s = t.empty(self.n_det, dtype=t.float64, device=self.device)
        _check(self.h, lib().chim_debug_injection_weights(self.h, self._lam1(lam).data_ptr(), s.data_ptr()))
        return s.cpu().numpy()
