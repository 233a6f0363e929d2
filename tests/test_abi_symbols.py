"""CPU-only: libchim.so loads and exports every symbol include/chim.h declares (no compute calls)."""
import ctypes
import os
import re
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "chim.h")


def _declared():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(chim_[a-z_]+)\s*\(", src)))


def test_header_is_plain_c():
    subprocess.run(["gcc", "-std=c99", "-Wall", "-Werror", "-fsyntax-only", "-x", "c", HEADER], check=True)
    src = re.sub(r"/\*.*?\*/", "", open(HEADER).read(), flags=re.S)      # signatures only, comments stripped
    assert 'extern "C"' in src and "torch" not in src.lower() and "at::" not in src and "std::" not in src


def test_library_exports_every_declared_symbol():
    import __graft_entry__ as g
    g.build()
    import paper_2504_02034_b200 as pkg
    lib = ctypes.CDLL(pkg.lib_path())
    names = _declared()
    assert {"chim_create", "chim_init_events", "chim_init_injections", "chim_loglike_batch", "chim_loglike_batch_host",
            "chim_destroy", "chim_last_error", "chim_version", "chim_get_stats"} <= set(names)
    for n in names:
        assert hasattr(lib, n), n
    assert pkg.chim_version() == 100


def test_default_config_and_no_device_failure():
    import paper_2504_02034_b200 as pkg
    cfg = pkg.chim_default_config()
    assert (cfg.kde_cutoff, cfg.z_cat_max, cfg.z_table_max) == (6.0, 1.5, 10.0)
    assert (cfg.n_table, cfg.n_dl_table, cfg.n_win_table, cfg.lambda_chunk) == (2048, 0, 512, 1024)
    assert cfg.placement == pkg.CHIM_ON_SAMPLES and cfg.bw_rule == pkg.CHIM_BW_SCOTT
    import torch
    if not torch.cuda.is_available():
        with pytest.raises(pkg.ChimError):          # no CPU fallback: creating a context without a GPU fails loudly
            pkg.chim_create(cfg)
        with pytest.raises(pkg.ChimError):
            pkg.Context()


def test_product_never_imports_the_oracle():
    pkgdir = os.path.join(ROOT, "paper_2504_02034_b200")
    for dp, _, fs in os.walk(pkgdir):
        for f in fs:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dp, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "chim_oracle" not in txt, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert "paper_2504_02034_b200" not in txt.replace("paper_2504_02034_b200/csrc", "").replace(
                "shares nothing with paper_2504_02034_b200", ""), f
