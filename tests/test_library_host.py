"""CPU-only checks of the C-ABI library: it loads, exports every symbol include/spin.h declares, its host
logic (argument validation, buffer sizes, threshold tables) is right, and it fails loudly without a GPU."""
import ctypes
import math
import os
import re

import numpy as np
import pytest

import paper_2304_01772_b200 as sp
from paper_2304_01772_b200 import binding

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "spin.h")).read()
    return sorted(set(re.findall(r"SPIN_API[^;(]*?\b(spin_[a-z_]+)\s*\(", text)))


def test_library_exports_every_declared_symbol():
    lib = sp.load_library()
    declared = _declared_symbols()
    assert len(declared) >= 16
    assert sorted(binding.EXPORTED_SYMBOLS) == declared
    for name in declared:
        assert getattr(lib, name) is not None


def test_no_torch_types_in_header():
    text = open(os.path.join(ROOT, "include", "spin.h")).read()
    assert "torch" not in text.lower().replace("pytorch", "") and "at::" not in text and "extern \"C\"" in text


def test_buffer_bytes():
    assert sp.spin_buffer_bytes(4, 32, sp.SPIN_MODEL_ISING, sp.SPIN_LAYOUT_INT8) == 4 * 32 * 32
    assert sp.spin_buffer_bytes(4, 8192, sp.SPIN_MODEL_ISING, sp.SPIN_LAYOUT_BITPACKED) == 4 * 8192 * 8192 // 8
    assert sp.spin_buffer_bytes(128, 512, sp.SPIN_MODEL_POTTS, sp.SPIN_LAYOUT_INT8) == 128 * 512 * 512
    assert sp.spin_buffer_bytes(1, 7, 0, 0) == 0          # odd L
    assert sp.spin_buffer_bytes(0, 8, 0, 0) == 0          # empty batch
    assert sp.spin_buffer_bytes(1, 32, 0, 1) == 0         # bit-packed needs L % 64 == 0
    assert sp.spin_buffer_bytes(1, 64, 1, 1) == 0         # bit-packed Potts


def test_threshold_table_equals_oracle_table(oracle_mod):
    # "compare threshold tables first": the library's host table vs the oracle's, bit for bit
    rng = np.random.default_rng(0)
    betas = list(rng.uniform(0.0, 3.0, 200)) + [0.0, 0.44, 0.4407, 20.0, 1e-12] + \
            [0.30 + 0.30 * b / 63.0 for b in range(64)]
    for beta in betas:
        for J, h in [(1.0, 0.0), (1.0, 0.01), (-1.0, 0.3), (0.7, -0.2)]:
            T, a = sp.spin_threshold_table(sp.SPIN_MODEL_ISING, beta, J, h)
            To, ao = oracle_mod.ising_table(beta, J, h)
            assert np.array_equal(a, ao) and np.array_equal(T[~a], To[~ao])
        for J in (1.0, -0.5):
            T, a = sp.spin_threshold_table(sp.SPIN_MODEL_POTTS, beta, J)
            To, ao = oracle_mod.potts_table(beta, J)
            assert np.array_equal(a, ao) and np.array_equal(T[~a], To[~ao])


def test_threshold_table_rejects_bad_arguments():
    for bad in (float("nan"), float("inf"), -0.1):
        with pytest.raises(sp.SpinError):
            sp.spin_threshold_table(sp.SPIN_MODEL_ISING, bad, 1.0, 0.0)
    with pytest.raises(sp.SpinError):
        sp.spin_threshold_table(7, 0.4, 1.0, 0.0)


def test_create_argument_validation_messages():
    for args, word in [((0, 8, 2, 1), "batch"), ((1, 7, 2, 1), "even"), ((1, 0, 2, 1), "even"),
                       ((1, 8, 1, 1), "q"), ((1, 8, 128, 1), "q")]:
        with pytest.raises(sp.SpinError) as e:
            sp.spin_create(*args)
        assert word in str(e.value)
    with pytest.raises(sp.SpinError) as e:
        sp.spin_create_ex(1, 64, sp.SPIN_MODEL_POTTS, q_uniform=3, layout=sp.SPIN_LAYOUT_BITPACKED)
    assert "Ising only" in str(e.value)
    with pytest.raises(sp.SpinError) as e:
        sp.spin_create_ex(1, 32, sp.SPIN_MODEL_ISING, layout=sp.SPIN_LAYOUT_BITPACKED)
    assert "64" in str(e.value)
    with pytest.raises(sp.SpinError):
        sp.spin_create_ex(2, 8, sp.SPIN_MODEL_POTTS, q_per_replica=[3, 200])
    with pytest.raises(sp.SpinError):
        sp.spin_create_ex(2, 8, sp.SPIN_MODEL_ISING, replica_offset=-1)


def test_null_handle_calls_fail_cleanly():
    lib = sp.load_library()
    assert lib.spin_sweep(None, None, 1.0, 0.0, 1, 0) == sp.SPIN_ERR_INVALID
    assert lib.spin_observables(None, None, None) == sp.SPIN_ERR_INVALID
    assert lib.spin_get_spins(None, None) == sp.SPIN_ERR_INVALID
    assert lib.spin_kernel_launches(None) == 0
    lib.spin_destroy(None)  # no-op


def test_fails_loudly_without_gpu():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(sp.SpinError) as e:
        sp.spin_create(4, 32, 2, 1)
    assert "no CPU fallback" in str(e.value)


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2304_01772_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "from oracle" not in text and "liboracle" not in text
                assert "spin_oracle" not in text


def test_workload_recipes():
    w = sp.workloads.config(2)
    assert (w.batch, w.L, w.n_sweeps, w.seed) == (64, 1024, 2000, 2)
    assert w.beta[0] == 0.30 and abs(w.beta[-1] - 0.60) < 1e-15
    w = sp.workloads.config(4)
    assert list(w.q[:64]) == [3] * 64 and list(w.q[64:]) == [8] * 64
    assert abs(w.beta[0] - 0.5 * math.log(1 + math.sqrt(3))) < 1e-15
    assert abs(w.beta[127] - 1.5 * math.log(1 + math.sqrt(8))) < 1e-15
    w = sp.workloads.config(5)
    assert w.batch == 1024 and w.beta[0] == 0.2 and abs(w.beta[-1] - 0.7) < 1e-15 and w.therm == 2000
    assert sp.workloads.config(1).updates == 4096000 and sp.workloads.config(3).L == 8192
