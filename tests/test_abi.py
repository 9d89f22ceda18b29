"""CPU-side checks of the boundary: the C-ABI library builds for sm_100a, loads, and exports every
symbol include/rc.h declares; the binding's table matches the header; no compute call is made."""
import ctypes as C
import re
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parent.parent
HEADER = (ROOT / "include" / "rc.h").read_text()


def declared_symbols():
    return sorted(set(re.findall(r"\b(rc_[a-z_A-Z]+)\s*\(", HEADER)))


def test_header_declares_the_four_north_star_calls():
    for name in ("rc_create", "rc_set_atmosphere", "rc_solve_J", "rc_destroy"):
        assert name in declared_symbols()


def test_library_builds_and_exports_every_declared_symbol():
    from paper_2408_14425_b200 import binding, build
    lib_path = build.build()
    lib = C.CDLL(str(lib_path))
    for name in declared_symbols():
        assert hasattr(lib, name), f"{name} declared in include/rc.h but not exported by {lib_path.name}"
    assert set(binding.SYMBOLS) == set(declared_symbols())


def test_library_is_sm100a_and_uses_no_legacy_tensor_or_fallback_code():
    import shutil
    import subprocess
    from paper_2408_14425_b200 import build
    cuobjdump = shutil.which("cuobjdump") or "/usr/local/cuda/bin/cuobjdump"
    out = subprocess.run([cuobjdump, "-lelf", str(build.build())], capture_output=True, text=True).stdout
    assert "sm_100a" in out, out


def test_calls_without_a_device_fail_loudly():
    """No GPU here (or a non-sm_100 one) => rc_create returns RC_ERR_NO_DEVICE; nothing falls back to CPU."""
    import torch
    from paper_2408_14425_b200 import binding
    if torch.cuda.is_available() and torch.cuda.get_device_capability(0)[0] == 10:
        pytest.skip("an sm_100 device is present")
    with pytest.raises(binding.RcError) as e:
        binding.RadianceCascades(5)
    assert e.value.code == -3


def test_bad_config_is_rejected_before_touching_the_device():
    from paper_2408_14425_b200 import binding
    lib = binding.load()
    h = C.c_void_p()
    for cfg in (binding.rc_config(0, 1.0, 0, 0, 0), binding.rc_config(13, 1.0, 0, 0, 0),
                binding.rc_config(5, 0.0, 0, 0, 0), binding.rc_config(5, 1.0, 0, 3, 0)):
        assert lib.rc_create(C.byref(h), C.byref(cfg)) == -5
    assert lib.rc_create(None, None) == -1
    assert lib.rc_destroy(None) == -1
    assert lib.rc_workspace_bytes(None, 64, 64, 1, 0) == 0
    assert b"sm_100a" in lib.rc_version()
