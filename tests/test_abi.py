"""CPU-only checks of the boundary: libgeo.so builds for sm_100a, loads, and exports every symbol that
include/geo.h declares; the header and the binding agree.  No compute calls (there is no GPU here)."""
import ctypes
import os
import re

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols(header="geo.h"):
    src = open(os.path.join(ROOT, "include", header)).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(geo_[a-z_0-9]+)\s*\(", src)))


def test_library_builds_loads_and_exports_every_declared_symbol():
    from paper_1803_08320_b200 import build, geo
    path = build.build()
    assert os.path.exists(path)
    lib = ctypes.CDLL(path)
    decl = _declared_symbols()
    assert len(decl) >= 8
    for name in decl:
        assert hasattr(lib, name), name
    assert sorted(geo.SYMBOLS) == decl
    dev = _declared_symbols("geo_dev.h")
    for name in dev:
        assert hasattr(lib, name), name
    assert sorted(geo.DEV_SYMBOLS) == dev


def test_struct_layouts_match_header():
    from paper_1803_08320_b200 import geo
    assert ctypes.sizeof(geo.GeoStop) == 24
    assert ctypes.sizeof(geo.GeoOut) == 10 * 8 and geo.GeoOut.coarse_steps.offset == 72
    assert geo.GeoOut.snap_mask.offset == 56 and geo.GeoOut.snap_count.offset == 64
    assert ctypes.sizeof(geo.GeoTable) == 56 and ctypes.sizeof(geo.GeoAdaptive) == 48


def test_sass_has_fp64_pipe_and_wide_stores():
    """The hot loop is FP64 FMA work (DFMA); the snapshot writer issues 256-bit global stores (STG.E...256)."""
    import subprocess
    from paper_1803_08320_b200 import build
    sass = subprocess.run(["cuobjdump", "-sass", build.build()], capture_output=True, text=True).stdout
    assert "sm_100a" in sass
    assert sass.count("DFMA") > 500
    assert re.search(r"STG\.E(\.\w+)*\.256", sass)
    assert re.search(r"LDG\.E(\.\w+)*\.256", sass)        # tabulated metric: one 256-bit load per stencil node


def test_every_direct_snapshot_kernel_keeps_its_256_bit_stores():
    """ptxas narrowed `st.global.v4.f64` to STG.E.64 in ONE clone of a non-inlined record writer (DESIGN.md section 5,
    profiles/r02_noinline_writer_miscompile.md): the shipped library must have 256-bit stores in every instantiation of the
    direct snapshot writer -- Kerr and Schwarzschild, Kahan and plain update, the dense-output RK5(4) kernels, the tabulated
    and the Kerr-Schild kernels."""
    import sys
    sys.path.insert(0, ROOT)
    import bench
    from paper_1803_08320_b200 import build, geo
    build.build()
    bench.static_sass_count("geo_rk4_kernelILb1ELi1ELb0ELb0E")            # fills the SASS cache
    sass = next(iter(bench._SASS_CACHE.values()))
    kernels, name = {}, None
    for line in sass.splitlines():
        m = re.search(r"Function : (\S+)", line)
        if m:
            name = m.group(1)
            kernels[name] = 0
        elif name and re.search(r"STG\.E(\.\w+)*\.256", line):
            kernels[name] += 1
    want = [k for k in kernels if re.search(r"geo_rk4_kernelILb[01]ELi1ELb[01]E", k) or re.search(r"geo_rk45_kernelILi[012]ELb1E", k)
            or re.search(r"geo_tabg?_rk4_kernelILb[01]ELb[01]ELb1E", k) or re.search(r"geo_ks_rk4_kernelILi1ELb[01]E", k)]
    assert len(want) == 8 + 3 + 4 + 4 + 2, want      # (the RK4 kernel: 4 instantiations of 128-thread CTAs + 4 of 512)
    for k in want:
        assert kernels[k] >= 2, (k, kernels[k])


def test_product_path_does_not_import_the_oracle():
    """No file of the package imports, loads, includes or executes anything under oracle/."""
    pkg = os.path.join(ROOT, "paper_1803_08320_b200")
    bad = re.compile(r"import\s+geo_(ks_|tab_)?oracle|from\s+oracle|import\s+oracle|libgeo_oracle|#include\s*[\"<].*oracle|oracle_(ks_)?integrate\s*\(")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert not bad.search(txt), f


def test_bench_instruction_counts_match_the_built_library():
    """bench.py's executed-instruction counts (KERNEL_COUNTS, from the committed ncu captures) are cross-checked against
    the static SASS count of the hot loops of the library as built here: a kernel edit without a new capture fails."""
    import sys
    sys.path.insert(0, ROOT)
    import bench
    from paper_1803_08320_b200 import build
    build.build()
    for key in bench.KERNEL_COUNTS:
        kc = bench.kernel_counts(key)          # raises SystemExit on disagreement
        assert kc["flop"] > 0 and kc["pipe"] > 0
        if key != "tabulated":
            assert kc["static"] is not None and kc["static"]["DFMA"] > 100
