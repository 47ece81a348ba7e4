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


def _shingles(text, k=4):
    """runs of k consecutive code lines, whitespace removed, type keywords dropped and identifiers folded to one letter (so that a
    renamed copy still matches); comment-only and trivial lines (braces, short statements) are skipped"""
    import re
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    lines = []
    for ln in text.splitlines():
        ln = ln.split("//")[0]
        ln = re.sub(r"\b(const|double|float|int|long|unsigned|static|complex)\b", "", ln)
        ln = re.sub(r"[A-Za-z_][A-Za-z_0-9]*", "v", ln)
        ln = re.sub(r"\s+", "", ln)
        if len(ln) >= 8:
            lines.append(ln)
    return {tuple(lines[i:i + k]) for i in range(len(lines) - k + 1)}


def test_no_routine_of_the_checker_is_restated_in_the_product():
    """VERDICT r1 'What's weak' 1: the CUDA path and the checker share no code -- not even a transliterated
    routine.  Mechanical form: no four consecutive non-trivial statements of oracle/sf_oracle.c reappear, up to
    whitespace and identifier names, in any source file of the product."""
    ora = _shingles((ROOT / "oracle" / "sf_oracle.c").read_text())
    for f in sorted((ROOT / "paper_2301_01145_b200" / "csrc").iterdir()):
        common = ora & _shingles(f.read_text())
        assert not common, f"{f.name} restates checker code: {sorted(common)[:2]}"


def test_null_plan_calls_fail_without_a_device():
    import paper_2301_01145_b200 as sf

    L = sf.lib()
    assert L.sf_solve(None) == sf.SF_ERR_INVALID_ARG
    assert L.sf_get_output(None, 0, 0, None, 0) == sf.SF_ERR_INVALID_ARG
    assert L.sf_plan_destroy(None) == sf.SF_OK
    assert sf.sf_last_launch_count(None) == 0
