"""CPU-side checks of the boundary and the host logic: the C-ABI library builds and exports every
symbol include/srp.h declares, the ctypes structs match the header, the product fails loudly
without a GPU, the input recipes are sane, and the multi-rank sharding logic works under gloo."""
import ctypes
import os
import re
import subprocess
import sys

import numpy as np
import pytest

from paper_2602_10712_b200 import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def libpath():
    from paper_2602_10712_b200.build import build_library
    return build_library()


def test_library_exports_every_declared_symbol(libpath):
    hdr = open(os.path.join(ROOT, "include", "srp.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(srp_[a-z_0-9]+)\s*\(", hdr))
    assert {"srp_build_designs", "srp_forces", "srp_create", "srp_get_stats"} <= declared
    L = ctypes.CDLL(libpath)
    for name in declared:
        assert hasattr(L, name), name
    from paper_2602_10712_b200 import binding
    assert set(binding.EXPORTS) == declared


def test_struct_layouts_match_header():
    from paper_2602_10712_b200 import binding
    assert ctypes.sizeof(binding.srp_stats) == 8 * (6 + 16 + 2 + 4 + 4 + 1 + 3)
    assert ctypes.sizeof(binding.srp_options) == 48
    assert binding.srp_options.leaf_max.offset == 36 and binding.srp_options.bvh_builder.offset == 40
    assert binding.srp_options.primary_mode.offset == 24
    assert binding.srp_options.sampler.offset == 8


def test_host_constants_without_gpu(libpath):
    from paper_2602_10712_b200 import binding
    L = binding.load_library()
    for fam, T in W.TRI_COUNT.items():
        assert L.srp_family_tri_count(fam) == T
        assert L.srp_family_n_params(fam) == W.N_PARAMS[fam]
    assert L.srp_family_tri_count(9) == -1


def test_product_fails_loudly_without_gpu(libpath):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    from paper_2602_10712_b200 import binding
    with pytest.raises(RuntimeError):
        binding.Context(0)
    h = ctypes.c_void_p()
    assert binding.load_library().srp_create(ctypes.byref(h), 0, None) != 0      # C level: no fallback either


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2602_10712_b200")
    for dp, _, fs in os.walk(pkg):
        for f in fs:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dp, f)).read()
                assert not re.search(r"import\s+oracle|from\s+oracle|srp_oracle|libsrp_oracle|oracle/srp", src), f


def test_input_recipes():
    s = W.fibonacci_sphere(1024)
    assert s.dtype == np.float32 and np.allclose(np.linalg.norm(s, axis=1), 1, atol=1e-6)
    assert np.abs(s.mean(0)).max() < 1e-3
    f = W.fibonacci_sphere(64, True)
    assert (f[:, 2] > 0).all()
    for name, cfg in W.CONFIGS.items():
        th = cfg.params()
        assert th.shape == (cfg.D, W.N_PARAMS[cfg.family]) and th.dtype == np.float32
        assert np.array_equal(th, cfg.params())                         # seeded
    t2 = W.CONFIGS["cfg2_boxwing"].params()
    assert t2[:, 0].min() >= 2 and t2[:, 0].max() <= 8 and t2[:, 1].min() >= 0 and t2[:, 1].max() <= np.pi
    assert [c.primaries for c in W.CONFIGS.values()] == [1 << 22, 1 << 36, 1 << 36, 1 << 36, 1 << 32]
    assert len(W.icosphere(2)) == 320


def test_latlong_force_map_layout():
    """lat-long image of directions; unit vectors, rows = polar angle, north row first, and the
    pixel solid angles sin(theta) dtheta dphi sum to 4 pi."""
    d = W.latlong_directions(6, 12).reshape(6, 12, 3).astype(np.float64)
    assert np.allclose(np.linalg.norm(d, axis=2), 1.0, atol=1e-6)
    assert np.all(d[0, :, 2] > 0.9) and np.all(d[-1, :, 2] < -0.9)
    assert np.allclose(d[:, 0, 1] / d[:, 0, 0], np.tan(np.pi / 12), atol=1e-5)       # first column: phi = pi / 12
    assert np.allclose(d[2, :, 2], np.cos(np.pi * 2.5 / 6), atol=1e-6)
    th = np.pi * (np.arange(400) + 0.5) / 400
    assert abs((np.sin(th) * (np.pi / 400) * 2 * np.pi).sum() - 4 * np.pi) < 1e-4


def test_bench_reference_arm_contract():
    """`bench.py --impl reference` (the oracle on the host cores) prints ONE JSON line with the contract's keys."""
    import json
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    out = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--impl", "reference", "--workload",
                          "cfg1_plate", "--steps", "1", "--warmup", "1"], capture_output=True, text=True, timeout=300)
    assert out.returncode == 0, out.stderr
    lines = [l for l in out.stdout.splitlines() if l.strip()]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["metric"] == "photon-bounce segments/s" and d["unit"] == "segments/s"
    assert d["value"] > 0 and d["higher_is_better"] is True and d["n_gpus"] == 1 and d["steps"] == 1
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["value"] == d["value"]
    assert d["e2e"] == {"value": d["value"], "unit": "segments/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert d["config"]["workload"] == "cfg1_plate" and d["vs_baseline"] is None
