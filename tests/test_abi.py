"""CPU-side checks of the C-ABI boundary: the library builds, loads and exports every symbol that
include/pact.h declares; the Python record mirrors the C struct.  No compute calls (no GPU here)."""
import ctypes as C
import re
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parents[1]


@pytest.fixture(scope="module")
def pact_lib():
    from paper_1709_02733_b200 import build, binding
    build.build()
    return binding.lib()


def _declared_symbols():
    text = (ROOT / "include" / "pact.h").read_text()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(pact_[a-z_]+)\s*\(", text)))


def test_header_symbols_are_exported(pact_lib):
    from paper_1709_02733_b200 import binding
    declared = _declared_symbols()
    assert "pact_create" in declared and "pact_forward" in declared and "pact_adjoint" in declared
    assert sorted(binding.SYMBOLS) == declared
    for name in declared:
        assert hasattr(pact_lib, name), name


def test_params_struct_layout():
    from paper_1709_02733_b200.binding import PactParams
    # int nx,ny,nz ; (pad) double h, dt ; int nt, npml ; double pml_R, pml_cref, pml_beta_max
    assert PactParams.nx.offset == 0 and PactParams.nz.offset == 8
    assert PactParams.h.offset == 16 and PactParams.dt.offset == 24
    assert PactParams.nt.offset == 32 and PactParams.npml.offset == 36
    assert PactParams.pml_R.offset == 40 and C.sizeof(PactParams) == 64


def test_strerror_and_null_safety(pact_lib):
    assert pact_lib.pact_strerror(0) == b"ok"
    for code in range(-6, 0):
        assert pact_lib.pact_strerror(code) not in (b"", b"unknown error")
    pact_lib.pact_destroy(None)                      # NULL is allowed
    assert pact_lib.pact_device_bytes(None) == 0
    # argument validation happens before any CUDA call, so these work without a GPU
    h = C.c_void_p()
    assert pact_lib.pact_create(C.byref(h), None, None, None, None, None, None, 0, None) == -1
    assert pact_lib.pact_forward(None, None, None) == -1
    assert pact_lib.pact_adjoint(None, None, None) == -1
    assert pact_lib.pact_set_option(None, b"profile", 1) == -1


def test_no_oracle_in_product_path():
    """The product never imports or links the oracle (and the oracle never imports the product)."""
    pkg = ROOT / "paper_1709_02733_b200"
    for f in list(pkg.rglob("*.py")) + list(pkg.rglob("*.cu")) + list(pkg.rglob("*.cuh")):
        if f.name == "synth.py":
            continue   # input generators: docstring mentions both consumers, imports neither
        assert "oracle" not in f.read_text().lower(), f
    for f in (ROOT / "oracle").glob("*"):
        if f.suffix in (".py", ".c"):
            t = f.read_text()
            assert "binding" not in t and "libpact" not in t and "ctypes.CDLL(\"libpact" not in t, f


def test_sass_uses_tma_mbarriers_and_tensor_memory(pact_lib):
    """The built library's step kernels carry the sm_100a instructions the design rests on:
    TMA tensor loads completing on mbarriers, tensor-memory stores / loads (tcgen05.st / ld) and packed fp32 math —
    and nothing was compiled for another architecture."""
    import shutil
    import subprocess
    from paper_1709_02733_b200 import build
    tool = shutil.which("cuobjdump") or "/usr/local/cuda/bin/cuobjdump"
    if not Path(tool).exists():
        pytest.skip("cuobjdump not installed")
    sass = subprocess.run([tool, "-sass", str(build.LIB)], capture_output=True, text=True, check=True).stdout
    archs = set(re.findall(r"arch = (sm_\w+)", sass))
    assert archs == {"sm_100a"}, archs
    kernels = {}
    for chunk in sass.split("Function : ")[1:]:
        name = chunk.split("\n", 1)[0].strip()
        kernels[name] = chunk
    step = {n: c for n, c in kernels.items() if "k_step" in n}
    assert len(step) == 6, sorted(step)                      # elastic and fluid-only, C-PML-free / forward / adjoint
    for n, c in step.items():
        assert c.count("UTMALDG") >= 10, n                   # cp.async.bulk.tensor
        assert "SYNCS.ARRIVE.TRANS64" in c and "SYNCS.PHASECHK" in c, n      # mbarrier expect_tx / try_wait
        assert "FFMA2" in c, n                               # packed f32x2 arithmetic
    for n, c in step.items():
        if "acoustic" not in n:                              # elastic step kernels: tensor memory as per-thread scratch
            assert "STTM" in c and "LDTM" in c, n
