"""The C-ABI library loads on a CPU-only box and exports every symbol include/pvf.h declares;
host-side configuration logic (no GPU compute calls)."""
import ctypes as C
import os
import re

import pytest

import __graft_entry__ as entry
import paper_2602_19959_b200 as pkg
from paper_2602_19959_b200.binding import pvf_config


@pytest.fixture(scope="module")
def lib():
    entry.build()
    return pkg.load_library()


def _declared_symbols(repo_root, header="pvf.h"):
    text = open(os.path.join(repo_root, "include", header)).read()
    return re.findall(r"PVF_API\s+[\w\s\*]+?\b(pvf_\w+)\s*\(", text)


def test_every_declared_symbol_is_exported(lib, repo_root):
    names = _declared_symbols(repo_root)
    assert len(names) >= 15
    assert sorted(names) == sorted(pkg.EXPORTS)
    for n in names:
        assert getattr(lib, n) is not None
    # every header under include/ is covered: the diagnostic entry points exist in every build flavour
    import glob
    assert sorted(os.path.basename(h) for h in glob.glob(os.path.join(repo_root, "include", "*.h"))) == ["pvf.h", "pvf_debug.h"]
    dbg = _declared_symbols(repo_root, "pvf_debug.h")
    assert sorted(dbg) == ["pvf_debug_fc_prof", "pvf_debug_unet_prof"]
    for n in dbg:
        assert getattr(lib, n) is not None
    # and nothing is exported that no header declares
    import subprocess
    out = subprocess.run(["nm", "-D", "--defined-only", pkg.LIB_PATH], capture_output=True, text=True).stdout
    exported = sorted(l.split()[-1] for l in out.splitlines() if " T " in l and l.split()[-1].startswith("pvf_"))
    assert exported == sorted(names + dbg)


def test_header_cites_the_paper(repo_root):
    text = open(os.path.join(repo_root, "include", "pvf.h")).read()
    assert "PAPER.md" in text and "extern \"C\"" in text
    assert "torch" not in text.lower().replace("pytorch", "")


def test_default_config_and_workspace_bytes(lib):
    cfg = pkg.default_config(lib, 16000, 3_100_000)
    assert (cfg.n_intervals, cfg.n_bins, cfg.fc_in, cfg.fc_hidden, cfg.hist_channels) == (40, 100, 9, 25, 8)
    assert (cfg.k_e1, cfg.k_e2, cfg.k_b, cfg.k_d2, cfg.k_d1) == (25, 15, 5, 15, 25)
    assert cfg.unet_channels == 64 and cfg.max_peaks == 32 and cfg.peak_halfwidth == 3
    assert abs(cfg.peak_threshold - 0.01) < 1e-8 and abs(cfg.bin_width_mm - 0.1) < 1e-8
    nbytes = lib.pvf_workspace_bytes(C.byref(cfg))
    hist = 16000 * 40 * 800 * 4
    assert hist < nbytes < hist + 200 * 2**20          # pool = histogram + small scratch
    small = pkg.default_config(lib, 1, 40)
    assert 0 < lib.pvf_workspace_bytes(C.byref(small)) < 8 * 2**20   # below the paper's 16 MB arena
    withio = pkg.default_config(lib, 16000, 3_100_000, enable_host_io=1)
    assert lib.pvf_workspace_bytes(C.byref(withio)) > nbytes + 16000 * 4000 * 4


@pytest.mark.parametrize("field,value", [("n_intervals", 41), ("n_bins", 64), ("unet_channels", 48), ("k_e1", 27),
                                         ("max_peaks", 16), ("precision", 7), ("max_events", 0), ("max_tracks", 0), ("max_tracks", 1 << 29),
                                         ("split_mask", 64), ("split_mask", 1), ("fc_hidden", 32)])
def test_invalid_config_is_rejected_on_the_host(lib, field, value):
    # (split_mask 1 is the e1 split of the TF32 and FP16 modes; the default precision here is FP32, where no split exists)
    cfg = pkg.default_config(lib, 4, 100)
    setattr(cfg, field, value)
    assert lib.pvf_workspace_bytes(C.byref(cfg)) == 0
    h = C.c_void_p()
    from paper_2602_19959_b200.binding import _weights_struct
    from pvf_inputs import make_weights
    ws, keep = _weights_struct(make_weights("rand", 1))
    assert lib.pvf_create(C.byref(ws), C.byref(cfg), C.byref(h)) == pkg.PVF_ERR_CONFIG
    assert not h.value


def test_null_arguments(lib):
    assert lib.pvf_workspace_bytes(None) == 0
    assert lib.pvf_create(None, None, None) == pkg.PVF_ERR_ARG
    assert lib.pvf_destroy(None) == pkg.PVF_ERR_ARG
    assert lib.pvf_run(None, None, 0, None, None, None) == pkg.PVF_ERR_ARG
    assert lib.pvf_status_string(0) == b"PVF_OK" and lib.pvf_status_string(3) == b"PVF_ERR_CAPACITY"
    assert b"sm_100a" in lib.pvf_build_info()


def test_struct_sizes_match_header():
    # int32 x2, float x2, int32 x4, int32 x5, float x2, int32 x5, int64, int32 x3, float, int32 x2
    assert C.sizeof(pvf_config) == 112


def test_e1_split_is_a_mode_of_the_ten_bit_formats_only(lib):
    """split_mask = 1: accepted with PVF_PREC_TF32 and PVF_PREC_FP16 (a workspace size comes back), rejected with BF16 / FP32."""
    for prec, ok in (("tf32", True), ("fp16", True), ("bf16", False), ("fp32", False)):
        cfg = pkg.default_config(lib, 4, 100, precision=pkg.PRECISIONS[prec], split_mask=1)
        assert (lib.pvf_workspace_bytes(C.byref(cfg)) > 0) == ok, prec
