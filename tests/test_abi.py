"""CPU-only: the C-ABI library loads and exports every symbol include/ledds.h declares; the
parameter checks that need no GPU behave as documented."""
import ctypes as C
import os
import re

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _lib():
    import __graft_entry__ as g
    g.build()
    return C.CDLL(os.path.join(ROOT, "paper_2512_04997_b200", "libledds.so"))


def test_every_declared_symbol_is_exported():
    hdr = open(os.path.join(ROOT, "include", "ledds.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    names = sorted(set(re.findall(r"\b(ledds_[a-z0-9_]+)\s*\(", hdr)))
    assert len(names) >= 15
    lib = _lib()
    for n in names:
        assert hasattr(lib, n), n


def test_binding_names_match_header():
    import paper_2512_04997_b200 as L
    hdr = open(os.path.join(ROOT, "include", "ledds.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    names = set(re.findall(r"\b(ledds_[a-z0-9_]+)\s*\(", hdr))
    assert names == set(L.EXPORTS)
    for n in names - {"ledds_lbm_current"}:
        assert callable(getattr(L, n)), n
    assert "sm_100a" in L.ledds_version()


def test_struct_layouts_match_header_sizes():
    # ctypes mirrors vs. what the C compiler lays out for include/ledds.h
    import subprocess, tempfile
    import paper_2512_04997_b200 as L
    src = '#include <stdio.h>\n#include "ledds.h"\nint main(){printf("%zu %zu %zu\\n", sizeof(ledds_lbm_params), sizeof(ledds_dem_params), sizeof(ledds_cpl_params));return 0;}\n'
    with tempfile.TemporaryDirectory() as d:
        open(os.path.join(d, "s.c"), "w").write(src)
        subprocess.check_call(["gcc", "-I", os.path.join(ROOT, "include"), os.path.join(d, "s.c"), "-o", os.path.join(d, "s")])
        sizes = [int(v) for v in subprocess.check_output([os.path.join(d, "s")]).split()]
    assert sizes == [C.sizeof(L.LbmParams), C.sizeof(L.DemParams), C.sizeof(L.CplParams)]


def test_parameter_validation_without_gpu():
    import paper_2512_04997_b200 as L
    import pytest
    p = L.lbm_params(dict(shape=(8, 8, 8), tau=0.6, bc=(0, 0, 0), u_wall=None))
    assert L.ledds_lbm_workspace_bytes(p) == 2 * 19 * 512 * 8
    assert L.ledds_lbm_workspace_bytes_f32(p) == 2 * 19 * 512 * 4
    p.variant = 2
    with pytest.raises(L.LeddsError):
        L.ledds_lbm_workspace_bytes_f32(p)                     # no such kernel variant
    with pytest.raises(L.LeddsError):
        L.ledds_lbm_workspace_bytes(p)
    p.variant = 0
    p.layout = 1
    with pytest.raises(L.LeddsError):
        L.ledds_lbm_workspace_bytes(p)                         # two-lattice is the only layout
    p.layout = 0
    p.tau = 0.5
    with pytest.raises(L.LeddsError):
        L.ledds_lbm_workspace_bytes(p)
    d = dict(n=10, lo=(0, 0, 0), hi=(1, 1, 1), bc=(1, 1, 1), cell=0.1, dt=1e-3, g=(0, 0, 0), density=1.0, kn=1.0, kt=0.3,
             restitution=0.9, mu=0.1, max_contacts=16)
    sb, hb = L.ledds_dem_workspace_bytes(L.dem_params(d))
    assert sb > 0 and hb >= 2 * (10 * 4 + 10 * 16 * 4 + 10 * 16 * 24)
    d["bc"] = (0, 1, 1); d["cell"] = 0.4                      # periodic axis with only 2 cells
    with pytest.raises(L.LeddsError):
        L.ledds_dem_workspace_bytes(L.dem_params(d))
    d["max_contacts"] = 64
    with pytest.raises(L.LeddsError):
        L.ledds_dem_workspace_bytes(L.dem_params(d))
    d.update(max_contacts=16, bc=(1, 1, 1), n=0)               # an empty system is valid and needs no history
    sb0, hb0 = L.ledds_dem_workspace_bytes(L.dem_params(d))
    assert hb0 == 0 and sb0 > 0
    d["n"] = -1
    with pytest.raises(L.LeddsError):
        L.ledds_dem_workspace_bytes(L.dem_params(d))


def test_no_load_is_hoisted_above_the_dependent_launch_wait():
    """The kernels of a DEM step are chained by programmatic dependent launch: a kernel may start while its
    predecessor still runs and must not read what that one writes before `griddepcontrol.wait` (ACQBULK in SASS).  The
    compiler is free to hoist loads through `const __restrict__` pointers (LDG.E.CONSTANT) above the wait -- it did so
    once, for a block-uniform load, and the kernel read a word its predecessor had not written yet.  This checks the
    machine code of every kernel that waits: no global / generic load, atomic or reduction before the wait."""
    import shutil, subprocess
    _lib()
    obj = os.path.join(ROOT, "paper_2512_04997_b200", "csrc", "dem.o")
    tool = shutil.which("cuobjdump") or "/usr/local/cuda/bin/cuobjdump"
    sass = subprocess.run([tool, "-sass", obj], capture_output=True, text=True, check=True).stdout
    waits, fn, seen, early = 0, None, False, {}
    for line in sass.splitlines():
        m = re.search(r"Function : (\S+)", line)
        if m:
            fn, seen = m.group(1), False
            continue
        if fn is None:
            continue
        if "ACQBULK" in line:
            waits += not seen
            seen = True
        elif not seen and re.search(r"\b(LDG|LD\.E|ATOMG|ATOM\.|REDG|RED\.)", line):
            early.setdefault(fn, []).append(line.strip())
    assert waits >= 10                                        # the chain: hist, passes, scans, scatter, ranges, gather, detect, fill, force ...
    hoisted = {f: v for f, v in early.items() if "ACQBULK" in sass.split("Function : " + f, 1)[1].split("Function : ", 1)[0]}
    assert not hoisted, hoisted
    # the single-launch step exchanges data between its phases through global memory, with cluster barriers in between:
    # none of its loads may be of the non-coherent kind (which the compiler may move across a barrier and the L1 may
    # serve from a stale line)
    clusters = 0
    for body in sass.split("Function : ")[1:]:
        if "UCGABAR" in body:
            clusters += 1
            assert ".CONSTANT" not in body, body.split("\n", 1)[0]
    assert clusters >= 8                                      # T x HERTZ x PERIODIC
