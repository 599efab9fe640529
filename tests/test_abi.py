"""The C-ABI library builds for sm_100a, loads without a GPU and exports every symbol include/vlasov.h declares;
argument checks that need no device."""
import ctypes as C
import os
import re

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "vlasov.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(vlasov_[a-z_0-9]+)\s*\(", src)))


def test_header_declares_the_north_star_entry_points():
    names = _declared()
    for n in ("vlasov_init", "vlasov_step", "vlasov_moments", "vlasov_set_boundary"):
        assert n in names


def test_library_builds_loads_and_exports_every_declared_symbol():
    from paper_1406_5445_b200 import build, binding
    path = build.build()
    assert os.path.exists(path)
    L = C.CDLL(path)
    for n in _declared():
        assert hasattr(L, n), n
    assert sorted(binding.EXPORTS) == _declared()


def test_sass_is_sm100a_only():
    import subprocess
    from paper_1406_5445_b200 import build
    out = subprocess.run(["cuobjdump", "-lelf", build.build()], capture_output=True, text=True).stdout
    archs = set(re.findall(r"sm_(\d+a?)", out))
    assert archs == {"100a"}, archs


def test_argument_checks_without_a_device():
    from paper_1406_5445_b200 import binding
    from paper_1406_5445_b200 import inputs
    w = inputs.landau_workload()
    w.species[0].f_inf = 1.0
    sp = binding.make_species(w.species)
    cfg = binding.make_config(w.nx, w.ny, 0, 1, w.lx, w.ly, 0, 0)
    n = binding.vlasov_scratch_bytes(cfg, sp)
    assert n >= w.nx * w.ny * 64 * 8 * 8 * 8 and n % 128 == 0
    bad = binding.make_config(w.nx, 0, 0, 1, w.lx, w.ly, 0, 0)
    assert binding.vlasov_scratch_bytes(bad, sp) == 0
    w.species[0].nv = (64, 8, 7)                       # an odd count is as good as an even one
    assert binding.vlasov_scratch_bytes(cfg, binding.make_species(w.species)) > 0
    w.species[0].nv = (64, 8, 0)
    assert binding.vlasov_scratch_bytes(cfg, binding.make_species(w.species)) == 0
    assert binding.strerror(binding.ESHIFT).startswith("y shift")
    # null context -> EINVAL, never a crash
    assert binding.lib().vlasov_step(None, 0.1, None, None, 31) == binding.EINVAL
    assert binding.lib().vlasov_check(None) == binding.EINVAL
