"""The C-ABI libraries load on a machine without a GPU and export every function include/*.h declares;
the Python bindings' symbol lists are exactly the headers' (no compute call is made here)."""
import ctypes
import os
import re

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared(header, prefix):
    src = open(os.path.join(ROOT, "include", header)).read()
    src = re.sub(r"/\*.*?\*/", " ", src, flags=re.S)                       # drop comments
    src = re.sub(r"//[^\n]*", " ", src)
    names = set(re.findall(r"\b(%s\w+)\s*\(" % prefix, src))
    assert names, header
    return names


def test_libmg_exports_everything_mg_h_declares():
    from paper_2009_02702_b200 import build, mg
    names = _declared("mg.h", "mg_")
    lib = ctypes.CDLL(build.lib_path("libmg.so"))
    for n in sorted(names):
        assert hasattr(lib, n), f"libmg.so does not export {n}"
    assert set(mg.SYMBOLS) == names
    for n in mg.SYMBOLS:                                                   # every binding has its argtypes set
        assert getattr(mg.lib, n).argtypes is not None, n


def test_libmg_builder_exports_everything_mg_builder_h_declares():
    from paper_2009_02702_b200 import build, builder
    names = _declared("mg_builder.h", "mgb_")
    lib = ctypes.CDLL(build.lib_path("libmg_builder.so"))
    for n in sorted(names):
        assert hasattr(lib, n), f"libmg_builder.so does not export {n}"
    assert set(builder.SYMBOLS) == names


def test_no_device_means_an_error_code_not_a_fallback():
    """Without a CUDA device mg_load_graph must fail with MG_ERR_CUDA / MG_ERR_OOM (no CPU path exists)."""
    import numpy as np
    import pytest
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    from paper_2009_02702_b200 import mg
    z = np.zeros(2, np.uint32)
    with pytest.raises(mg.MgError) as ei:
        mg.Graph(z, z, np.zeros(2, np.float32), 2, level_offsets=np.array([0, 2], np.uint64))
    assert ei.value.code in (mg.MG_ERR_CUDA, mg.MG_ERR_OOM)


def test_reference_arm_workload_does_not_map_the_cuda_library():
    """bench.py --impl reference assembles its inputs with the generator and the host builder only (load=False): the
    binding of libmg.so is imported lazily, so that arm's process never maps the product's CUDA library."""
    import subprocess
    import sys
    code = ("import sys; from paper_2009_02702_b200 import workload; w = workload.make(1, load=False, device_synth=False); "
            "assert w.graph is None and w.host_graph['child_a'].size > 16; "
            "assert 'paper_2009_02702_b200.mg' not in sys.modules; "
            "assert 'libmg.so' not in open('/proc/self/maps').read(); print('ok')")
    out = subprocess.run([sys.executable, "-c", code], cwd=ROOT, capture_output=True, text=True, timeout=600)
    assert out.returncode == 0 and out.stdout.strip() == "ok", out.stderr[-2000:]
