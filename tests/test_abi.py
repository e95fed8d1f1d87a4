"""The C-ABI library loads and exports every symbol include/routebalance.h declares (no compute: no GPU here)."""
import ctypes
import os
import re

from conftest import ROOT


def _declared():
    """Every function include/*.h declares (routebalance.h: the decision API; routebalance_testing.h: the timing and
    self-test entry points of the tests and bench.py)."""
    names = set()
    inc = os.path.join(ROOT, "include")
    for h in sorted(os.listdir(inc)):
        if h.endswith(".h"):
            src = re.sub(r"/\*.*?\*/", "", open(os.path.join(inc, h)).read(), flags=re.S)
            names |= set(re.findall(r"\b(rb_[a-z_0-9]+)\s*\(", src))
    return sorted(names)


def test_library_builds_and_exports_declared_symbols():
    from paper_2606_17949_b200 import build
    lib = ctypes.CDLL(build.build())
    names = _declared()
    assert "rb_create" in names and "rb_decide" in names and len(names) >= 12
    for n in names:
        assert hasattr(lib, n), "librouteb.so does not export %s" % n


def test_binding_names_match_header():
    from paper_2606_17949_b200 import binding
    for n in _declared():
        assert hasattr(binding, n), "binding lacks %s" % n
    assert sorted(binding.EXPORTS) == _declared()


def test_options_default_and_null_handling_without_gpu():
    from paper_2606_17949_b200 import binding as rb
    o = rb.rb_options_default()
    assert (o.store_dtype, o.rerank_slack, o.lpt_enabled, o.update_enabled, o.max_batch, o.use_graph) == \
        (rb.RB_BF16, 6, 1, 1, 4096, 1)
    assert abs(o.dist_eps - 1e-6) < 1e-12
    rb.rb_destroy(None)                       # NULL is allowed
    assert rb._lib.rb_sync(None) == rb.RB_EINVAL
    assert rb.rb_launch_count(None) == 0


def test_product_never_imports_oracle():
    """The product path must not route through the oracle (or any CPU fallback): no file of the package
    imports, includes, links or loads anything under oracle/."""
    pkg = os.path.join(ROOT, "paper_2606_17949_b200")
    bad = re.compile(r"(from\s+oracle|import\s+oracle|oracle\.orc|import\s+orc\b|liborc|orc\.cpp|#include\s+\"[^\"]*oracle)")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                text = open(os.path.join(dirpath, f)).read()
                assert not bad.search(text), "%s references the oracle" % f
    for f in ("orc.cpp", "orc.py"):
        text = open(os.path.join(ROOT, "oracle", f)).read()
        assert not re.search(r"(import\s+paper_2606|from\s+paper_2606\S*\s+import|#include\s+\"[^\"]*(csrc|routebalance))", text), f


def test_c_program_links_and_runs(tmp_path):
    """include/routebalance.h is valid C99 and librouteb.so links from a plain C program (no Python, no torch):
    defaults, argument validation and NULL handling through the C ABI, without a GPU."""
    import subprocess
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    pkg = os.path.join(root, "paper_2606_17949_b200")
    exe = str(tmp_path / "abi_check")
    subprocess.run(["gcc", "-std=c99", "-Wall", "-Werror", "-I", os.path.join(root, "include"),
                    os.path.join(pkg, "examples", "abi_check.c"), "-o", exe, "-L", pkg, "-lrouteb",
                    "-Wl,-rpath," + pkg], check=True)
    r = subprocess.run([exe], capture_output=True, text=True)
    assert r.returncode == 0 and "abi ok" in r.stdout, (r.returncode, r.stdout, r.stderr)
