"""vlasov_fluid_step_static (include/vlasov.h): the fluid step of section 3.2 for callers that cannot
allocate device memory -- its Runge-Kutta stage buffers sit in a static device array of the library (4 MiB).  Checked
against the existing entry point vlasov_fluid_step (caller's scratch; itself checked against oracle/fluid.py in
test_gpu_fluid.py) on two calls in a row that share the array, of different shapes, so the second call finds the first
one's leftovers.  Collected last on purpose (file name): the suite runs with pytest -x."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu
TOL = 1e-12            # the tolerance of test_gpu_fluid.py; the two entry points run the same kernels, so also bitwise


@pytest.fixture(scope="module")
def gpu():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1406_5445_b200 import binding
    binding.lib()
    return binding


def dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def rough_state(rng, ns, ny, nx):
    U = np.zeros((ns, 5, ny + 4, nx))
    for s in range(ns):
        rho = 1.0 + 0.5 * rng.random((ny + 4, nx))
        rho[ny // 2:, : nx // 2] *= 3.0
        v = 0.6 * (rng.random((3, ny + 4, nx)) - 0.5)
        p = 0.8 + 0.4 * rng.random((ny + 4, nx))
        U[s, 0] = rho
        U[s, 1:4] = rho[None] * v
        U[s, 4] = 1.5 * p + 0.5 * rho * (v ** 2).sum(0)
    return U


def one_case(gpu, seed, ns, ny, nx, bc, steps):
    import torch
    rng = np.random.default_rng(seed)
    q = [-1.0, 1.0, 2.0][:ns]
    m = [0.04, 1.0, 4.0][:ns]
    U0 = rough_state(rng, ns, ny, nx)
    E = 0.3 * rng.standard_normal((3, ny + 4, nx))
    B = 0.5 * rng.standard_normal((3, ny + 4, nx))
    gl = gh = None
    if bc == gpu.FLUID_BC_COUPLED:
        gl = dev(rough_state(rng, 3 * ns, -2, nx).reshape(3, ns, 5, 2, nx))
        gh = dev(rough_state(rng, 3 * ns, -2, nx).reshape(3, ns, 5, 2, nx))
    blk = gpu.FluidBlock(nx, ny, 0.11, 0.13, q, m, bc, bc)
    Ed, Bd = dev(E), dev(B)
    Ua, Ub = dev(U0), dev(U0)
    for _ in range(steps):
        blk.vlasov_fluid_step(0.004, Ua, Ed, Bd, gl, gh)             # existing path: caller's scratch
        blk.vlasov_fluid_step_static(0.004, Ub, Ed, Bd, gl, gh)      # new path: the library's static array
    torch.cuda.synchronize()
    want, got = Ua.cpu().numpy()[:, :, 2:-2], Ub.cpu().numpy()[:, :, 2:-2]
    assert np.isfinite(got).all()
    assert np.abs(want - U0[:, :, 2:-2]).max() > 1e-3                # the step did something
    assert np.linalg.norm((got - want).ravel()) <= TOL * np.linalg.norm(want.ravel())
    assert np.abs(got - want).max() <= TOL * np.abs(want).max()
    assert np.array_equal(got, want)


def test_static_scratch_step_matches_the_callers_scratch_step_on_two_calls_in_a_row(gpu):
    # first call: a block that fills 2.1 of the 4 MiB (config 4's fluid blocks: 2 species on 256 x 48), coupled sides
    one_case(gpu, 71, 2, 48, 256, gpu.FLUID_BC_COUPLED, steps=2)
    # second call: another shape, species count and boundary kind on top of the first call's leftovers
    one_case(gpu, 72, 3, 7, 9, gpu.FLUID_BC_WALL, steps=3)
    one_case(gpu, 73, 1, 16, 32, gpu.FLUID_BC_PERIODIC, steps=2)


def test_static_scratch_step_refuses_blocks_beyond_its_maximum(gpu):
    import torch
    ns, ny, nx = 2, 100, 256                                        # 2 * 104 * 256 = 53248 cells > 52428
    blk = gpu.FluidBlock(nx, ny, 0.1, 0.1, [-1.0, 1.0], [1.0, 1.0], gpu.FLUID_BC_WALL, gpu.FLUID_BC_WALL)
    assert blk.scratch.numel() > gpu.FLUID_STATIC_SCRATCH_BYTES
    U = torch.ones((ns, 5, ny + 4, nx), dtype=torch.float64, device="cuda")
    Z = torch.zeros((3, ny + 4, nx), dtype=torch.float64, device="cuda")
    with pytest.raises(gpu.VlasovError) as e:
        blk.vlasov_fluid_step_static(0.01, U, Z, Z)
    assert e.value.code == gpu.ETOOBIG and "static scratch" in str(e.value)
    assert bool((U == 1.0).all())                                   # nothing was launched
    ok = gpu.FluidBlock(nx, 98, 0.1, 0.1, [-1.0, 1.0], [1.0, 1.0], gpu.FLUID_BC_WALL, gpu.FLUID_BC_WALL)   # the largest that fits
    assert ok.scratch.numel() <= gpu.FLUID_STATIC_SCRATCH_BYTES
    U = torch.ones((ns, 5, 98 + 4, nx), dtype=torch.float64, device="cuda")
    U[:, 4] = 3.0
    Z = torch.zeros((3, 98 + 4, nx), dtype=torch.float64, device="cuda")
    ok.vlasov_fluid_step_static(0.01, U, Z, Z)
    torch.cuda.synchronize()
    assert bool(torch.isfinite(U).all())
    with pytest.raises(gpu.VlasovError) as e:                       # the checks of vlasov_fluid_step still apply
        gpu.FluidBlock(4, 4, 0.1, 0.1, [1.0], [1.0], gpu.FLUID_BC_COUPLED, gpu.FLUID_BC_COUPLED).vlasov_fluid_step_static(
            0.01, torch.ones((1, 5, 8, 4), dtype=torch.float64, device="cuda"), Z, Z)
    assert e.value.code == gpu.EINVAL
