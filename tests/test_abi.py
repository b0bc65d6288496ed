"""The C-ABI boundary on a CPU box: libepw_interp.so loads, exports every function include/epw_interp.h declares, the
Python binding lists exactly those, and the product refuses to run without a GPU (no CPU fallback, no oracle behind it)."""
import ctypes
import os
import re
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

HEADER = os.path.join(ROOT, "include", "epw_interp.h")


def declared_functions():
    text = open(HEADER).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)  # drop comments
    names = re.findall(r"\b(epw_[a-z0-9_]+)\s*\(", text)
    return sorted(set(names))


@pytest.fixture(scope="module")
def lib():
    from paper_2603_10295_b200 import build

    return ctypes.CDLL(build.build_library())


def test_header_declares_the_contract_entry_points():
    names = declared_functions()
    for must in ("epw_interp_create", "epw_interp_set_wannier_operators", "epw_interp_interpolate", "epw_interp_destroy",
                 "epw_interp_interpolate_grid", "epw_phase_table", "epw_rp_to_q", "epw_eigh_batched", "epw_zgemm",
                 "epw_rotate_g2", "epw_wannier_from_bloch", "epw_interp_set_energy_window", "epw_interp_set_rp_shard"):
        assert must in names


def test_library_exports_every_declared_symbol(lib):
    missing = [n for n in declared_functions() if not hasattr(lib, n)]
    assert not missing, f"declared in include/epw_interp.h but not exported: {missing}"


def test_binding_lists_exactly_the_declared_symbols():
    from paper_2603_10295_b200 import binding

    assert sorted(binding.EXPORTED_SYMBOLS) == declared_functions()
    for n in binding.EXPORTED_SYMBOLS:   # and wraps each of them under the same name (or a class method for create/destroy)
        assert hasattr(binding, n), f"binding.py has no wrapper called {n}"


def test_no_cpu_fallback():
    """Without a CUDA device every compute entry fails loudly; nothing routes to oracle/."""
    import torch

    if torch.cuda.is_available():
        pytest.skip("this check is for the CPU box")
    import paper_2603_10295_b200 as epw

    with pytest.raises(epw.EpwError) as e:
        epw.epw_interp_create(8, 6, 27, 27)
    assert e.value.code == epw.binding.EPW_ECUDA
    src = open(os.path.join(ROOT, "paper_2603_10295_b200", "binding.py")).read()
    assert "import oracle" not in src and "from oracle" not in src
    for f in os.listdir(os.path.join(ROOT, "paper_2603_10295_b200", "csrc")):
        assert "oracle" not in open(os.path.join(ROOT, "paper_2603_10295_b200", "csrc", f)).read().replace(
            "Nothing in here is used by oracle/", "")


def test_create_rejects_a_negative_or_nan_omega_min():
    """Argument validation happens before the device is touched, so it is checkable on a CPU box: a negative cut-off
    would let soft modes (reported with negative omega) into 1/sqrt(2 omega)."""
    import paper_2603_10295_b200 as epw

    for bad in (-1e-3, float("nan")):
        with pytest.raises(epw.EpwError) as e:
            epw.epw_interp_create(8, 6, 27, 27, omega_min=bad)
        assert e.value.code == epw.binding.EPW_EINVAL
        assert "omega_min" in str(e.value)


def test_bench_host_logic_without_a_gpu():
    """bench.py imports on a CPU box, its per-config defaults are the ones the full-size parity tests use, and the record
    it keeps of an extra config is built from the fields run_config() produces."""
    import bench

    assert bench.NQ_STEP[1] == 96 and bench.NQ_STEP[2] == 32 and bench.NQ_STEP[3] == 13 and bench.NQ_STEP[4] == 2
    sub = {"config": {"workload": "w", "k_side": "cached after warm-up: H(k) ...", "cold_call_ms": 2.5}, "value": 1.0, "unit": "elements/s", "ms_per_step": 2.0, "steps": 3, "warmup": 1,
           "gpu_launches": 7, "clocks": {"sm_mhz": 1965.0},
           "roofline": {"stage": "S4b_rotate_g2", "kernel": "k", "bound": "tensor", "achieved": 1.0, "peak": 2.0,
                        "unit": "TFLOP/s", "frac": 0.5, "share_of_step": 0.4, "traffic": None,
                        "stages": {"S1_rp_to_q": {"kernel": "rp_to_q_kernel", "bound": "hbm", "frac": 0.7, "share_of_step": 0.04}}},
           "klist_path": {"value": 3.0, "ms_per_step": 4.0, "S2_re_to_k": {"kernel": "zgemm_dmma_kernel", "bound": "tensor",
                                                                          "frac": 0.96, "share_of_step": 0.8}},
           "parity": {"ok": True, "pairs": 96, "worst_g2_over_tolerance": 0.123456789}}
    rec = bench.summarise_config(sub, 1.5)
    assert rec["k_side"] == "cached after warm-up" and rec["cold_call_ms"] == 2.5
    # the compact summary that goes LAST into the JSON line: three configs and the consumer figure within 1,200 characters
    import json

    sub["value"], sub["ms_per_step"] = 3.123456789e10, 16.123456
    sub["roofline"]["kernel"] = "rotate_g2_tma_kernel (two-kernel form)"
    sub["roofline"]["stages"]["S4b_rotate_g2"] = {"kernel": "rotate_g2_tma_kernel", "frac": 0.4812345}
    sub["clocks"] = {"sm_mhz": 1965.0, "sm_max_mhz": 1965.0, "reasons": ["sw_power_cap"]}
    recs = {str(i): bench.summarise_config(sub, 1.5) for i in (2, 3, 4)}
    brief = bench.brief_of(recs, {"value": 4.3e10, "ms": 56.3, "d2h_bytes_per_step": 8000000, "device_ms": 55.0})
    assert len(json.dumps(brief)) <= 1200, len(json.dumps(brief))
    assert brief["3"]["kernel"] == "rotate_g2_tma_kernel" and brief["3"]["s4b"] == 0.481 and brief["3"]["parity_ok"] is True
    assert brief["2"]["worst"] == 0.123 and brief["2"]["cold_ms"] == 2.5 and brief["e2e_consumer"]["ms"] == 56.3
    assert rec["dominant"]["frac"] == 0.5 and rec["stages"]["S1_rp_to_q"]["frac"] == 0.7
    assert rec["klist_path"]["S2_re_to_k"]["frac"] == 0.96 and rec["parity"]["ok"] and rec["wall_s"] == 1.5
