"""The C-ABI library builds without a GPU (nvcc cross-compiles), loads, and exports every symbol include/uts.h declares;
the Python binding lists the same names; host-only calls work; compute calls refuse CPU tensors (no CPU fallback)."""
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "uts.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(uts_[a-z_0-9]+)\s*\(", src)))


def test_library_exports_every_declared_symbol():
    from paper_2606_29794_b200 import build, binding as B
    build.build()
    L = B.lib()
    names = _declared()
    assert len(names) >= 17
    for n in names:
        assert hasattr(L, n), n
    assert sorted(B.SYMBOLS) == names
    for n in names:                     # the binding offers the same names
        if n not in ("uts_last_cuda_error", "uts_strerror", "uts_version"):
            assert hasattr(B, n), n


def test_host_only_calls_and_status_strings():
    from paper_2606_29794_b200 import binding as B
    L = B.lib()
    assert L.uts_version().decode().startswith("uts")
    assert L.uts_strerror(B.UTS_ERR_CAPACITY).decode() == "caller buffer too small"
    t = B.uts_rho_max_table()
    assert len(t) == 14 and abs(t[0] - 0.8410686705679302) < 1e-12 and all(a > b for a, b in zip(t, t[1:]))
    cfg = B.Config(order=10, n_gauss=2_000_000, sh_degree=3)
    assert B.uts_tile_query_scratch_bytes(cfg) > 4 * 2_000_000
    assert B.uts_sort_scratch_bytes(1_000_000) > 0
    assert B.uts_host_workspace_bytes(cfg, -1, 1000) > 2_000_000 * 236
    assert B.uts_tile_query_scratch_bytes(B.Config(order=3, n_gauss=1)) == 0      # order < tile_log2: invalid config


def test_no_cpu_fallback():
    import torch
    from paper_2606_29794_b200 import binding as B
    cfg = B.Config(order=6, n_gauss=4)
    z = torch.zeros(16)
    with pytest.raises(RuntimeError):
        B.uts_preprocess(cfg, B.Gaussians(z, z, z, z, z), B.Views(z, z), B.Proj(z, z, z, z, z, z, z.to(torch.uint8)))
    if not torch.cuda.is_available():
        from paper_2606_29794_b200 import rasterizer as R
        with pytest.raises(RuntimeError):
            R.Rasterizer(cfg)
