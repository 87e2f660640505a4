"""CPU-only checks of the boundary: the C-ABI library builds for sm_100a, loads, and exports
every symbol include/sph_b200.h declares; argument checks that need no GPU."""
import ctypes
import os
import re

from paper_1807_08116_b200 import binding

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "sph_b200.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(?:int|size_t|int64_t)\s+((?:sph|nbody)_\w+)\s*\(", src)))


def test_library_exports_every_declared_symbol():
    lib = binding.load()
    names = _declared()
    assert len(names) >= 18 and "nbody_pp_gravity" in names and "sph_step" in names
    for n in names:
        assert hasattr(lib, n), f"{n} declared in include/sph_b200.h but not exported"
    assert set(names) == set(binding.EXPORTS)


def test_north_star_entry_points_present():
    for n in ("sph_build_grid", "sph_neighbour_ranges", "sph_density", "sph_forces", "nbody_pp_gravity", "sph_step"):
        assert callable(getattr(binding, n))


def test_workspace_size_and_arg_checks_without_gpu():
    g = binding.sph_grid.make((0, 0, 0), 0.4, 2.5, (48, 48, 49))
    a = binding.sph_workspace_bytes(4096, 8192, g)
    b = binding.sph_workspace_bytes(8192, 16384, g)
    assert 0 < a < b
    lib = binding.load()
    assert lib.sph_workspace_bytes(10, 5, ctypes.byref(g)) == 0          # n_gas > n_total
    big = binding.sph_grid.make((0, 0, 0), 0.4, 2.5, (4097, 1, 1))
    assert lib.sph_workspace_bytes(10, 10, ctypes.byref(big)) == 0       # dimension > 4096
    # argument errors are reported before any CUDA call
    assert lib.nbody_pp_gravity(None, 10, 1.0, 0.1, None, None, 0, None) == binding.SPH_ERR_ARG
    assert lib.nbody_pp_gravity(None, 10, 1.0, -0.1, None, None, 0, None) == binding.SPH_ERR_UNSUPPORTED
    assert lib.nbody_pp_gravity(None, 0, 1.0, 0.1, None, None, 0, None) == binding.SPH_OK
    assert lib.sph_step_host(None, None, 1, 1, None, 0.1, 1, None, None, None) != binding.SPH_OK


def test_sass_is_blackwell_native():
    """The gravity kernel must contain packed FP32 math and a TMA bulk copy (sm_100a SASS)."""
    import shutil
    import subprocess
    cu = shutil.which("cuobjdump") or "/usr/local/cuda/bin/cuobjdump"
    if not os.path.exists(cu):
        return
    sass = subprocess.run([cu, "-sass", binding.lib_path()], capture_output=True, text=True).stdout
    assert "sm_100a" in sass
    for mnem in ("FFMA2", "FADD2", "FMUL2", "MUFU.RSQ", "UBLKCP"):
        assert mnem in sass, mnem


def test_gravity_sums_region_without_gpu():
    """sph_workspace_gravity_sums (host-only): the int64 region of the pair-symmetric path lies inside the workspace,
    256-byte aligned, 24 bytes per source padded to whole 2048-source blocks."""
    lib = binding.load()
    off, nb = ctypes.c_size_t(0), ctypes.c_size_t(0)
    g = binding.sph_grid.make((0, 0, 0), 0.4, 2.5, (48, 48, 49))
    for n_gas, n, grid in ((0, 100000, None), (4096, 8192, g), (0, 1, None), (0, 2048, None), (0, 2049, None)):
        gp = ctypes.byref(grid) if grid is not None else None
        assert lib.sph_workspace_gravity_sums(n_gas, n, gp, ctypes.byref(off), ctypes.byref(nb)) == 0
        assert nb.value == 24 * ((n + 2047) // 2048 * 2048) and off.value % 256 == 0
        assert off.value + nb.value <= lib.sph_workspace_bytes(n_gas, n, gp)
    assert lib.sph_workspace_gravity_sums(5, 3, None, ctypes.byref(off), ctypes.byref(nb)) == binding.SPH_ERR_ARG
    assert lib.sph_workspace_gravity_sums(5, 8, None, ctypes.byref(off), ctypes.byref(nb)) == binding.SPH_ERR_ARG   # gas needs a grid
    assert lib.sph_workspace_gravity_sums(0, 8, None, None, ctypes.byref(nb)) == binding.SPH_ERR_ARG


def test_concurrent_builds_do_not_corrupt_the_library():
    """torchrun ranks on a fresh checkout all call build() at once: each must compile into its own
    temporary and serialise on the lock, so that the library every one of them ends up loading is whole.  Exercised
    on the oracle's build (same pattern as csrc/build.py, seconds instead of half a minute)."""
    import subprocess
    import sys
    code = ("import sys; sys.path.insert(0, %r); from oracle.build import build; import ctypes; "
            "p = build(force=True); L = ctypes.CDLL(p); L.orc_rc2.restype = ctypes.c_float; "
            "L.orc_rc2.argtypes = [ctypes.c_float]; assert L.orc_rc2(1.0) == 4.0" % ROOT)
    procs = [subprocess.Popen([sys.executable, "-c", code]) for _ in range(4)]
    assert [p.wait(timeout=300) for p in procs] == [0, 0, 0, 0]
    left = [f for f in os.listdir(os.path.join(ROOT, "oracle")) if f.endswith(".tmp")]
    assert left == []
