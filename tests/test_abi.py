"""The C-ABI library builds for sm_100a without a GPU, loads, and exports every symbol that
include/sailffish.h declares (no compute calls here)."""
import ctypes
import re
from pathlib import Path

ROOT = Path(__file__).resolve().parent.parent


def _declared():
    text = (ROOT / "include" / "sailffish.h").read_text()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(sf_[a-z_0-9]+)\s*\(", text)))


def test_header_declares_the_north_star_calls():
    names = _declared()
    for need in ("sf_plan_create", "sf_set_source", "sf_set_bc_values", "sf_solve", "sf_gradient", "sf_curl",
                 "sf_get_output"):
        assert need in names


def test_library_builds_loads_and_exports_every_declared_symbol():
    from paper_2301_01145_b200 import _build
    import paper_2301_01145_b200 as sf

    lib_path = _build.build()
    assert lib_path.exists()
    L = ctypes.CDLL(str(lib_path))
    declared = _declared()
    assert sorted(sf.EXPORTS) == declared, "binding EXPORTS and header declarations differ"
    for name in declared:
        assert hasattr(L, name), f"{name} is declared in sailffish.h but not exported"
    L.sf_version.restype = ctypes.c_char_p
    assert b"sm_100a" in L.sf_version()


def test_binding_has_no_cpu_fallback_and_no_oracle_import():
    src = (ROOT / "paper_2301_01145_b200" / "__init__.py").read_text()
    assert "import oracle" not in src and "from oracle" not in src
    for f in (ROOT / "paper_2301_01145_b200" / "csrc").iterdir():
        assert "oracle" not in f.read_text().lower(), f"{f.name} mentions the oracle"


def test_null_plan_calls_fail_without_a_device():
    import paper_2301_01145_b200 as sf

    L = sf.lib()
    assert L.sf_solve(None) == sf.SF_ERR_INVALID_ARG
    assert L.sf_get_output(None, 0, 0, None, 0) == sf.SF_ERR_INVALID_ARG
    assert L.sf_plan_destroy(None) == sf.SF_OK
    assert sf.sf_last_launch_count(None) == 0
