"""The C-ABI library builds, loads without a GPU and exports every symbol include/ep.h declares."""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    txt = open(os.path.join(ROOT, "include", "ep.h")).read()
    txt = re.sub(r"/\*.*?\*/", "", txt, flags=re.S)
    return sorted(set(re.findall(r"\b(ep_[a-z0-9_]+)\s*\(", txt)))


def test_every_declared_symbol_is_exported_and_bound():
    import paper_2112_12854_b200 as ep
    from paper_2112_12854_b200.binding import SIGNATURES
    L = ep.lib()
    names = _declared()
    assert len(names) >= 25
    for n in names:
        assert hasattr(L, n), f"{n} declared in ep.h but not exported by libep.so"
        assert n in SIGNATURES, f"{n} declared in ep.h but not bound in binding.py"
    assert sorted(SIGNATURES) == names


def test_no_oracle_or_cpu_fallback_in_product():
    """The product path never imports or links the oracle."""
    pkg = os.path.join(ROOT, "paper_2112_12854_b200")
    for dp, _, fs in os.walk(pkg):
        for f in fs:
            if f.endswith((".py", ".cu", ".cuh", ".cpp", ".h")):
                src = open(os.path.join(dp, f)).read()
                assert "ep_oracle" not in src and "from oracle" not in src and "import oracle" not in src, f


def test_model_state_counts_match_paper():
    """TP06 has 19 state variables, Courtemanche 21."""
    import paper_2112_12854_b200 as ep
    assert ep.model_n_states(ep.EP_MODEL_TP06) == 19
    assert ep.model_n_states(ep.EP_MODEL_CRN98) == 21
    assert ep.model_n_states(99) < 0


def test_error_paths_need_no_gpu():
    import paper_2112_12854_b200 as ep
    L = ep.lib()
    assert L.ep_step(None, 1, 0.02) == -1
    assert b"null" in L.ep_last_error()
    xyz = np.array([[0, 0, 0], [1, 0, 0], [0, 1, 0], [0, 0, 1]], dtype=np.float64)
    with pytest.raises(ep.EpError) as e:   # index out of range
        ep.host_stencil(xyz, np.array([[0, 1, 2, 7]], dtype=np.int32))
    assert e.value.code == -2
    with pytest.raises(ep.EpError) as e:   # zero volume
        ep.host_stencil(np.array([[0, 0, 0], [1, 0, 0], [2, 0, 0], [3, 0, 0]], dtype=np.float64),
                        np.array([[0, 1, 2, 3]], dtype=np.int32))
    assert e.value.code == -2
    with pytest.raises(ep.EpError) as e:   # zero fibre
        ep.host_stencil(xyz, np.array([[0, 1, 2, 3]], dtype=np.int32), fibre=np.zeros((1, 3)))
    assert e.value.code == -2
    with pytest.raises(ep.EpError) as e:   # face shared by three cells
        x5 = np.array([[0, 0, 0], [1, 0, 0], [0, 1, 0], [0, 0, 1], [0, 0, -1], [1, 1, 1]], dtype=np.float64)
        ep.host_stencil(x5, np.array([[0, 1, 2, 3], [0, 1, 2, 4], [0, 1, 2, 5]], dtype=np.int32))
    assert e.value.code == -2
    with pytest.raises(ep.EpError) as e:   # bad sigma
        ep.host_stencil(xyz, np.array([[0, 1, 2, 3]], dtype=np.int32), sigma_l=-1.0)
    assert e.value.code == -1


def test_mesh_create_without_gpu_fails_loudly():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    import paper_2112_12854_b200 as ep
    xyz = np.array([[0, 0, 0], [1, 0, 0], [0, 1, 0], [0, 0, 1]], dtype=np.float64)
    with pytest.raises(ep.EpError) as e:
        ep.Sim(xyz, np.array([[0, 1, 2, 3]], dtype=np.int32))
    assert e.value.code == -4 and "no CPU fallback" in str(e.value)


def test_noalloc_entry_point_refuses_bad_sizes_without_a_gpu():
    """ep_weighted_mean_noalloc checks its arguments before any CUDA call: the size limit of its fixed scratch is an error
    that names the limit (include/ep.h: EP_NOALLOC_MAX_N)."""
    import paper_2112_12854_b200 as ep
    txt = open(os.path.join(ROOT, "include", "ep.h")).read()
    assert int(re.search(r"#define EP_NOALLOC_MAX_N (\d+)LL", txt).group(1)) == ep.NOALLOC_MAX_N == 8192 * 4096
    with pytest.raises(ep.EpError) as e:
        ep.weighted_mean_noalloc(8, 8, ep.NOALLOC_MAX_N + 1, 8)
    assert e.value.code == -1 and "EP_NOALLOC_MAX_N" in str(e.value) and str(ep.NOALLOC_MAX_N) in str(e.value)
    for args in ((0, 8, 8, 8), (8, 0, 8, 8), (8, 8, 8, 0), (8, 8, 0, 8), (8, 8, -3, 8)):
        with pytest.raises(ep.EpError) as e:
            ep.weighted_mean_noalloc(*args)
        assert e.value.code == -1
    src = open(os.path.join(ROOT, "paper_2112_12854_b200", "csrc", "ep_noalloc.cu")).read()
    code = re.sub(r"//.*", "", src)
    assert "cudaMalloc" not in code and "cudaFree" not in code and "cudaGetSymbolAddress" in code

