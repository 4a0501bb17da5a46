"""CPU-side checks of the boundary: the C-ABI library builds, loads and exports every symbol that
include/corr.h declares; the product never reaches into oracle/ (and vice versa); without a GPU
the compute entry points fail loudly instead of falling back."""
from __future__ import annotations

import ast
import os
import re
import shutil

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

needs_nvcc = pytest.mark.skipif(shutil.which("nvcc") is None and not os.path.exists(
    os.path.join(ROOT, "paper_0906_1887_b200", "libcorr.so")), reason="no nvcc and no prebuilt libcorr.so")


def header_symbols(name="corr.h"):
    text = open(os.path.join(ROOT, "include", name)).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(corr_[a-z0-9_]+)\s*\(", text)))


@needs_nvcc
def test_library_exports_every_declared_symbol():
    import paper_0906_1887_b200 as pkg
    L = pkg.lib()
    syms = header_symbols()
    assert {"corr_create", "corr_xengine", "corr_destroy"} <= set(syms)
    for s in syms:
        assert hasattr(L, s), f"{s} declared in include/corr.h but not exported"
    assert set(pkg.EXPORTS) == set(syms)
    # the diagnostics (include/corr_diag.h) live in libcorr_diag.so only: the product library carries neither the
    # probe entry points nor the probe-instrumented kernel instantiations
    diag = header_symbols("corr_diag.h")
    assert set(pkg.DIAG_EXPORTS) == set(diag) and {"corr_probe_mma", "corr_probe_ffma", "corr_set_probe"} <= set(diag)
    for s in diag:
        assert not hasattr(L, s), f"{s} is a diagnostic but libcorr.so exports it"
    D = pkg.diag_lib()
    for s in syms + diag:
        assert hasattr(D, s), f"{s} missing from libcorr_diag.so"


@needs_nvcc
def test_product_library_reads_no_environment_and_has_one_instantiation_per_kernel():
    """Plan knobs go through corr_set_option, not getenv; each hot kernel is instantiated once in libcorr.so."""
    import subprocess
    import paper_0906_1887_b200 as pkg
    pkg.lib()
    for f in os.listdir(os.path.join(ROOT, "paper_0906_1887_b200", "csrc")):
        assert "getenv" not in open(os.path.join(ROOT, "paper_0906_1887_b200", "csrc", f)).read(), f
    if shutil.which("cuobjdump") is None:
        pytest.skip("cuobjdump not available")
    lib = os.path.join(ROOT, "paper_0906_1887_b200", "libcorr.so")
    out = subprocess.run(["cuobjdump", "-elf", lib], capture_output=True, text=True, timeout=300).stdout
    names = set(re.findall(r"\.text\.(_ZN4corr\w+)", out))
    kernels = sorted(n for n in names if "xengine" in n or "fengine" in n)
    assert len(kernels) == 8, kernels   # i8, i8_batch, i8_pair, i4, f32, f32_n64, fengine, fengine_ci4
    assert not any("probe" in n for n in names), names


@needs_nvcc
def test_no_cpu_fallback_without_device():
    torch = pytest.importorskip("torch")
    if torch.cuda.is_available():
        pytest.skip("a device is present")
    import paper_0906_1887_b200 as pkg
    with pytest.raises(pkg.CorrError) as e:
        pkg.corr_create(64, 2, 10, "ci8")
    assert e.value.status in (pkg.CORR_ECUDA, pkg.CORR_EARCH)
    # argument validation happens before any device work and needs no GPU
    for bad in [(48, 2, 10, "ci8"), (64, 2, 70000, "ci8"), (64, 0, 10, "cf32")]:
        with pytest.raises(pkg.CorrError) as e:
            pkg.corr_create(*bad)
        assert e.value.status in (pkg.CORR_EINVAL, pkg.CORR_EUNSUPPORTED)
    L = pkg.lib()
    assert L.corr_destroy(None) == pkg.CORR_OK
    assert L.corr_xengine(None, None, None, None) == pkg.CORR_EINVAL
    assert L.corr_xengine_batch(None, None, None, 1, None) == pkg.CORR_EINVAL
    assert L.corr_set_option(None, pkg.CORR_OPT_PAIRS, 0) == pkg.CORR_EINVAL
    assert L.corr_set_chan_window(None, 4, 0) == pkg.CORR_EINVAL
    assert L.corr_accumulate_wide(None, None, None, None) == pkg.CORR_EINVAL
    assert L.corr_accumulate_count(None) == 0 and L.corr_acc_bytes(None) == 0
    # F-stage: same rules (no device -> error code; bad shapes rejected before any device work)
    with pytest.raises(pkg.CorrError) as e:
        pkg.corr_fstage_create(64, 128, 10)
    assert e.value.status in (pkg.CORR_ECUDA, pkg.CORR_EARCH)
    for bad in [(64, 64, 10), (48, 128, 10), (64, 128, 0)]:
        with pytest.raises(pkg.CorrError) as e:
            pkg.corr_fstage_create(*bad)
        assert e.value.status in (pkg.CORR_EINVAL, pkg.CORR_EUNSUPPORTED)
    assert L.corr_fstage_destroy(None) == pkg.CORR_OK
    assert L.corr_fstage_run(None, None, None, None) == pkg.CORR_EINVAL


def _imports(path):
    tree = ast.parse(open(path).read())
    names = set()
    for node in ast.walk(tree):
        if isinstance(node, ast.Import):
            names |= {a.name.split(".")[0] for a in node.names}
        elif isinstance(node, ast.ImportFrom) and node.module and node.level == 0:
            names.add(node.module.split(".")[0])
    return names


def test_product_and_oracle_are_independent():
    pkg_dir = os.path.join(ROOT, "paper_0906_1887_b200")
    for dirpath, _, files in os.walk(pkg_dir):
        for f in files:
            p = os.path.join(dirpath, f)
            if f.endswith(".py"):
                assert "oracle" not in _imports(p), f"{p} imports the oracle"
            if f.endswith((".cu", ".cuh", ".h", ".py")):
                assert "oracle/" not in open(p).read().replace("oracle/.", ""), f"{p} references oracle/"
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        p = os.path.join(ROOT, "oracle", f)
        if f.endswith(".py"):
            assert "paper_0906_1887_b200" not in _imports(p)
        if f.endswith((".c", ".h")):
            src = open(p).read()
            assert "#include \"../" not in src and "csrc" not in src
    # the generators hold none of the method's arithmetic and import neither side
    gen = _imports(os.path.join(ROOT, "corrgen", "__init__.py"))
    assert "oracle" not in gen and "paper_0906_1887_b200" not in gen
    # bench.py may use the oracle only in its cpu_baseline / reference legs
    bench = os.path.join(ROOT, "bench.py")
    if os.path.exists(bench):
        src = open(bench).read()
        for m in re.finditer(r"^\s*import oracle|^\s*from oracle", src, flags=re.M):
            pre = src[:m.start()]
            fn = re.findall(r"^def (\w+)", pre, flags=re.M)[-1]
            assert fn.startswith("cpu_baseline") or fn == "run_reference", f"bench.py imports oracle inside {fn}()"


@needs_nvcc
def test_sass_is_blackwell_native():
    """The built library carries tcgen05 MMAs (UTCIMMA, incl. the 2-CTA form), TMEM loads (LDTM) and TMA
    (UTMALDG) in its SASS, and no legacy tensor path (HMMA/IMMA warp-level MMAs)."""
    if shutil.which("cuobjdump") is None:
        pytest.skip("cuobjdump not available")
    import subprocess
    import paper_0906_1887_b200 as pkg
    pkg.lib()
    lib = os.path.join(ROOT, "paper_0906_1887_b200", "libcorr.so")
    sass = subprocess.run(["cuobjdump", "-sass", lib], capture_output=True, text=True, timeout=300).stdout
    assert "sm_100a" in sass
    for mnemonic in ("UTCIMMA", "UTCIMMA.2CTA", "LDTM", "UTMALDG", "UTCBAR"):
        assert mnemonic in sass, f"{mnemonic} missing from the SASS"
    assert " HMMA" not in sass and " IMMA" not in sass
