"""CPU-side checks of the boundary: the shared library loads, exports every symbol include/azint.h declares, and its
argument validation / error behaviour works without a GPU.  No compute calls here."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def B(cuda_lib):
    from paper_1412_6367_b200 import binding
    binding.lib()
    return binding


def _declared_functions():
    text = open(os.path.join(ROOT, "include", "azint.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(ai_[a-z0-9_]+)\s*\(", text)))


def test_library_exports_every_declared_symbol(B):
    names = _declared_functions()
    assert {"ai_setup", "ai_build_csr", "ai_get_csr", "ai_copy_csr_to_host", "ai_set_options", "ai_integrate1d", "ai_integrate1d_batch",
            "ai_integrate1d_host", "ai_destroy", "ai_strerror", "ai_last_error"} <= set(names)
    L = B.lib()
    for n in names:
        assert hasattr(L, n), f"{n} declared in include/azint.h but not exported"
    assert sorted(B.EXPORTS) == names


def test_binding_enums_match_header():
    text = open(os.path.join(ROOT, "include", "azint.h")).read()
    from paper_1412_6367_b200 import binding as B
    for name, val in re.findall(r"\b(AI_[A-Z0-9_]+)\s*=\s*(-?\d+)", text):
        assert getattr(B, name) == int(val), name


def test_setup_validation(B):
    def setup(**kw):
        a = dict(distance_m=0.1, pixel_y_m=1e-4, pixel_x_m=1e-4, center_y_px=8.0, center_x_px=8.0, wavelength_m=1e-10,
                 height=16, width=16, npt=10, unit=B.AI_R_MM, radial_range=None)
        a.update(kw)
        return B.ai_setup(**a)
    ctx = setup()
    assert ctx.value
    B.ai_destroy(ctx)
    for bad in (dict(npt=0), dict(height=0), dict(width=-3), dict(distance_m=0.0), dict(pixel_x_m=-1e-4),
                dict(wavelength_m=0.0), dict(unit=7), dict(radial_range=(2.0, 2.0)), dict(radial_range=(3.0, 1.0)),
                dict(center_x_px=float("nan")), dict(distance_m=float("inf"))):
        with pytest.raises(B.AzintError) as e:
            setup(**bad)
        assert e.value.code == B.AI_EINVAL, bad
    with pytest.raises(B.AzintError) as e:
        setup(height=70000, width=70000)
    assert e.value.code == B.AI_EUNSUPPORTED
    B.ai_destroy(C.c_void_p(None))      # NULL is allowed


def test_calls_before_build_are_refused(B):
    ctx = B.ai_setup(0.1, 1e-4, 1e-4, 8.0, 8.0, 1e-10, 16, 16, 10, B.AI_TTH_DEG)
    L = B.lib()
    assert L.ai_get_csr(ctx, None, None, None, None, None, None) == B.AI_ENOTBUILT
    dummy = C.c_void_p(16)
    assert L.ai_integrate1d(ctx, dummy, B.AI_F32, None, None, None, None, None, None, dummy, dummy, dummy, None) \
        == B.AI_ENOTBUILT
    assert L.ai_integrate1d_host(ctx, dummy, B.AI_F32, None, None, None, None, None, dummy, dummy, dummy, None) \
        == B.AI_ENOTBUILT
    assert b"ai_build_csr" in L.ai_last_error(ctx)
    assert L.ai_hold_corrections(ctx, dummy, None, None, None, None, None) == B.AI_ENOTBUILT
    assert L.ai_hold_corrections(ctx, None, None, None, None, None, None) == B.AI_ENOTBUILT
    assert L.ai_set_options(ctx, B.AI_LAYOUT_LUT, B.AI_ACC_F64, 1.5) == B.AI_OK
    assert L.ai_set_options(ctx, 5, 0, 0.0) == B.AI_EINVAL
    assert L.ai_last_launch_count(ctx) == 0
    B.ai_destroy(ctx)


def test_null_context_is_an_error_not_a_crash(B):
    L = B.lib()
    assert L.ai_build_csr(None, None) == B.AI_EINVAL
    assert L.ai_set_options(None, 0, 0, 0.0) == B.AI_EINVAL
    assert L.ai_hold_corrections(None, None, None, None, None, None, None) == B.AI_EINVAL
    assert L.ai_integrate1d(None, None, 0, None, None, None, None, None, None, None, None, None, None) == B.AI_EINVAL
    assert L.ai_strerror(B.AI_ECUDA) == b"CUDA error" and L.ai_strerror(123) == b"unknown status"
    assert L.ai_last_error(None) == b""


def test_no_cpu_fallback_without_a_gpu(B):
    import torch
    if torch.cuda.is_available():
        pytest.skip("this check is for the CPU-only box")
    ctx = B.ai_setup(0.1, 1e-4, 1e-4, 8.0, 8.0, 1e-10, 16, 16, 10, B.AI_R_MM)
    rc = B.lib().ai_build_csr(ctx, None)
    assert rc == B.AI_ECUDA and B.lib().ai_last_error(ctx) != b""       # fails loudly, computes nothing
    B.ai_destroy(ctx)
    from paper_1412_6367_b200 import workloads
    with pytest.raises(RuntimeError):
        B.Integrator(workloads.CONFIGS["cfg1"])


def test_setup2d_azimuthal_range_limits(B):
    """0 < chi1 - chi0 <= 2 pi inside [-2 pi, 3 pi] (include/azint.h): beyond 3 pi the builder's three images of a pixel
    (shifted by -2 pi, 0, +2 pi) would leave bins silently empty, so such a range is refused at set-up."""
    import math

    def setup(rng):
        return B.ai_setup2d(0.1, 1e-4, 1e-4, 8.0, 8.0, 1e-10, 16, 16, 5, 6, B.AI_R_MM, None, rng)
    for ok in ((-math.pi, math.pi), (0.0, 2 * math.pi), (-2 * math.pi, 0.0), (math.pi, 3 * math.pi), (0.5, 1.5)):
        B.ai_destroy(setup(ok))
    for bad in ((1.5 * math.pi, 3.5 * math.pi), (2 * math.pi, 4 * math.pi), (-2.5 * math.pi, -1.0), (0.0, 7.0),
                (1.0, 1.0), (2.0, 1.0), (0.0, float("nan"))):
        with pytest.raises(B.AzintError) as e:
            setup(bad)
        assert e.value.code == B.AI_EINVAL, bad


def test_path_options_are_an_explicit_call_not_the_environment(B):
    """The library reads no environment variable (plain C structs and enums): kernels are re-routed
    only through ai_set_path_options, before the matrix is built."""
    src = os.path.join(ROOT, "paper_1412_6367_b200", "csrc")
    for name in os.listdir(src):
        if name.endswith((".cu", ".cuh", ".h")):
            assert "getenv" not in open(os.path.join(src, name)).read(), name
    ctx = B.ai_setup(0.1, 1e-4, 1e-4, 8.0, 8.0, 1e-10, 16, 16, 10, B.AI_TTH_DEG)
    B.ai_set_path_options(ctx, force_fl=1, fl_chunk=2, fl_stages=2)
    B.ai_set_path_options(ctx)                                   # back to the defaults
    L = B.lib()
    assert L.ai_set_path_options(ctx, None) == B.AI_OK           # NULL = defaults
    for bad in (dict(no_fl=1, force_fl=1), dict(fl_chunk=-1), dict(fl_stages=-2)):
        with pytest.raises(B.AzintError) as e:
            B.ai_set_path_options(ctx, **bad)
        assert e.value.code == B.AI_EINVAL, bad
    opt = B.ai_path_options()
    opt.reserved[3] = 1
    assert L.ai_set_path_options(ctx, C.byref(opt)) == B.AI_EINVAL
    assert L.ai_set_path_options(None, None) == B.AI_EINVAL
    with pytest.raises(B.AzintError):
        B.ai_set_path_options(ctx, no_such_switch=1)
    B.ai_destroy(ctx)
