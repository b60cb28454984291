"""Parity of FULL pixel splitting (ai_set_splitting(AI_SPLIT_FULL)) on the CUDA path against the CPU
oracle (oracle/azint_oracle.c, pinned in tests/test_oracle_pins_full.py): the matrix and the per-bin results.
"""
import numpy as np
import pytest

from parity import assert_profile, compare_csr

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    return torch


@pytest.fixture(scope="module")
def B(cuda_lib):
    from paper_1412_6367_b200 import binding
    binding.lib()
    return binding


def _cases(W):
    return {
        "centred": W.tiny_config(96, 96, center_x=48.0, center_y=48.0, unit=W.R_MM, npt=60, name="centred"),
        "inside_a_pixel": W.tiny_config(80, 112, center_x=40.4, center_y=61.7, unit=W.TTH_DEG, npt=77, name="inside_a_pixel"),
        "off_image_q": W.tiny_config(67, 259, center_x=-12.5, center_y=300.0, unit=W.Q_NM, npt=301, name="off_image_q"),
        "narrow_bins": W.tiny_config(129, 65, center_x=32.0, center_y=64.0, unit=W.R_MM, npt=400, name="narrow_bins"),
        "cfg1b": W.CONFIGS["cfg1b"],
    }


def _dev(torch, a):
    return None if a is None else torch.from_numpy(np.ascontiguousarray(a)).cuda()


@pytest.mark.parametrize("name", ["centred", "inside_a_pixel", "off_image_q", "narrow_bins", "cfg1b", "cfg2"])
def test_full_splitting_matrix_and_profiles(torch, B, oracle, workloads, parity_report, name):
    cfg = workloads.CONFIGS["cfg2"] if name == "cfg2" else _cases(workloads)[name]
    integ = B.Integrator(cfg, split=B.AI_SPLIT_FULL)
    gi, gx, gd, (u0, u1) = integ.csr()
    oi, ox, od, (o0, o1) = oracle.csr_full(cfg)
    assert u0 == pytest.approx(o0, rel=1e-15, abs=1e-300) and u1 == pytest.approx(o1, rel=4e-16)
    # a corner exactly on a bin edge gives a zero-area slice on one side and none on the other: counted as ties
    rep = compare_csr((gi, gx, gd), (oi, ox, od), cfg.npix, max_ties=4 * (cfg.height + cfg.width))
    bbox = B.Integrator(cfg)                               # (kept alive while its context is read)
    bbox_nnz = int(B.ai_get_csr(bbox.ctx)[3])
    bbox.close()
    rep["nnz_bounding_box"] = bbox_nnz
    print(name, rep)
    assert rep["nnz_gpu"] <= bbox_nnz                      # the quadrilateral lies inside its bounding box
    parity_report.setdefault("full_splitting_csr_vs_oracle", {})[cfg.name] = rep
    # profiles: plain frame and a frame with every correction, tiled and canonical-CSR kernels
    rng = np.random.default_rng(51)
    shape = (cfg.height, cfg.width)
    img = workloads.make_frame(cfg).image if name in ("cfg1b", "cfg2") else rng.poisson(150.0, size=shape).astype(np.float32)
    frames = [workloads.Frame(image=img),
              workloads.Frame(image=img, dark=rng.poisson(5.0, size=shape).astype(np.float32),
                              flat=rng.uniform(0.9, 1.1, size=shape).astype(np.float32),
                              mask=(rng.random(shape) < 0.04).astype(np.uint8))]
    for layout in (B.AI_LAYOUT_TILED, B.AI_LAYOUT_CSR):
        integ.set_options(layout)
        for fr in frames:
            want = oracle.integrate1d_full(cfg, fr)
            args = [_dev(torch, x) for x in (fr.image, fr.dark, fr.flat, fr.solidangle, fr.polarization, fr.mask)]
            i, s, c = integ.integrate1d(*args)
            torch.cuda.synchronize()
            got = {"intensity": i.cpu().numpy(), "sum_signal": s.cpu().numpy(), "count": c.cpu().numpy()}
            assert_profile(got, want, what=f"full/{name}/{layout}")
    integ.close()


def test_splitting_is_fixed_once_built(torch, B, workloads):
    integ = B.Integrator(workloads.CONFIGS["cfg1"])
    with pytest.raises(B.AzintError):
        B.ai_set_splitting(integ.ctx, B.AI_SPLIT_FULL)
    integ.close()


def test_scatter_layout_is_refused_with_full_splitting(torch, B, workloads):
    """AI_LAYOUT_SCATTER splits by bounding box on the fly: on a context whose matrix was built with full pixel splitting
    it would silently disagree with every other layout, so the call is refused."""
    cfg = _cases(workloads)["centred"]
    integ = B.Integrator(cfg, split=B.AI_SPLIT_FULL)
    img = torch.ones((cfg.height, cfg.width), dtype=torch.float32, device="cuda")
    integ.set_options(layout=B.AI_LAYOUT_SCATTER)
    with pytest.raises(B.AzintError) as e:
        integ.integrate1d(img)
    assert e.value.code == B.AI_EUNSUPPORTED and "AI_SPLIT_FULL" in str(e.value)
    integ.set_options()
    i, s, c = integ.integrate1d(img)
    torch.cuda.synchronize()
    assert np.allclose(i.cpu().numpy()[c.cpu().numpy() > 0], 1.0, rtol=1e-6)
    integ.close()
