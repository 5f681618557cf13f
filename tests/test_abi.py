"""CPU-side checks of the boundary: the C-ABI library builds for sm_100a, loads, and exports every
symbol include/dgfs.h declares; argument validation that happens before any CUDA call.  No compute."""
import ctypes as C
import os
import re

import pytest

import __graft_entry__ as entry
from paper_1903_04670_b200 import api


@pytest.fixture(scope="module")
def lib():
    entry.build()
    return api.load_library()


def _declared_symbols(repo_root):
    src = open(os.path.join(repo_root, "include", "dgfs.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(dgfs_[a-z_0-9]+)\s*\(", src)))


def test_every_declared_symbol_is_exported(lib, repo_root):
    declared = _declared_symbols(repo_root)
    assert set(declared) == set(api.ABI_SYMBOLS), (declared, api.ABI_SYMBOLS)
    for name in declared:
        assert hasattr(lib, name), name
    assert sorted(api.exported_symbols()) == declared


def test_library_is_in_tree_and_has_sm100a_code(lib, repo_root):
    path = api.library_path()
    assert path.startswith(repo_root)
    import subprocess
    out = subprocess.run(["cuobjdump", "-lelf", path], capture_output=True, text=True).stdout
    assert "sm_100a" in out


def test_create_rejects_bad_arguments_before_touching_cuda(lib):
    # every case must fail in validation (EINVAL / ENOSUP), never reach the device probe
    good = dict(mass=[1.0, 2.0], omega=[0.5] * 4, alpha=[1.0] * 4, N=8, N_rho=4, M=6, L=5.0)

    def code(**kw):
        args = dict(good)
        args.update(kw)
        with pytest.raises(api.DgfsError) as e:
            api.dgfs_create(**args)
        return e.value.code, str(e.value)

    assert code(N=7)[0] == api.DGFS_EINVAL
    assert code(N=10)[0] == api.DGFS_ENOSUP
    assert code(mass=[1.0, -2.0])[0] == api.DGFS_EINVAL
    assert code(alpha=[1.0, 0.0, 1.0, 1.0])[0] == api.DGFS_EINVAL
    c, msg = code(omega=[0.5, 2.5, 0.5, 0.5])
    assert c == api.DGFS_EINVAL and "omega" in msg
    assert code(N_rho=0)[0] == api.DGFS_EINVAL
    assert code(L=-1.0)[0] == api.DGFS_EINVAL
    assert code(M=7)[0] == api.DGFS_EINVAL                      # no built-in rule, no sigma given
    assert code(table_mode=1)[0] == api.DGFS_EINVAL             # needs the pre-sphere
    import numpy as np
    sig = np.eye(3).repeat(2, axis=0) * np.array([1, -1, 1, -1, 1, -1])[:, None]
    assert code(sigma=sig, w_sigma=[1.0] * 6)[0] == api.DGFS_EINVAL   # weights do not sum to 4 pi
    assert code(sigma=sig * 1.1, w_sigma=[4 * np.pi / 6] * 6)[0] == api.DGFS_EINVAL


def test_no_cpu_fallback_without_device(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("CUDA device present")
    with pytest.raises(api.DgfsError) as e:
        api.dgfs_create([1.0], [0.5], [1.0], 8, 4, 6, 5.0)
    assert e.value.code == api.DGFS_ECUDA
    assert "no CPU fallback" in str(e.value)


def test_null_context_calls_fail_cleanly(lib):
    assert lib.dgfs_collide(None, None, None, 1, None) == api.DGFS_EINVAL
    assert lib.dgfs_collide_pairs(None, None, None, 1, None) == api.DGFS_EINVAL
    assert lib.dgfs_reserve(None, 1) == api.DGFS_EINVAL
    assert lib.dgfs_workspace_bytes(None, 1) == 0
    assert lib.dgfs_flops_per_pair_eval(None, 0, 0) == 0.0
    lib.dgfs_destroy(None)


def test_product_does_not_import_oracle(repo_root):
    pkg = os.path.join(repo_root, "paper_1903_04670_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, fn)).read()
                assert not re.search(r"(import|from)\s+oracle|oracle/", txt), os.path.join(dirpath, fn)
