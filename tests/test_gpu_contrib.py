"""GPU parity of the per-splat contribution C_k^V (Eq. 20-21) and the covisibility score (Eq. 22):
sgs_render_contrib / sgs_covisibility against oracle.contribution / oracle.covisibility.
C_k is a sum of blending coefficients: EVERY splat is compared at 1e-4 relative with an absolute floor of 1e-3 "pixels"
(the 24-bit fixed-point warp sum quantises each pixel's coefficient to 6e-8) plus the oracle-derived exposure of the
fragile pixels the splat touches (C_k is the colour gradient of sum_p I_r(p), so oracle.exposure of that upstream bounds
what a flipped decision can move); the covisibility counts are integer work and must match exactly on identical inputs."""
import numpy as np
import pytest
import torch

import oracle
import scenegen

pytestmark = pytest.mark.gpu

sgs = pytest.importorskip("paper_2506_00970_b200")
from gpu_common import to_device, camera, alloc_images, planes, C_EXPO  # noqa: E402


def gpu_contrib(ren, sf, n, cam, T_cw=None):
    c = camera(cam, T_cw)
    im = alloc_images(cam)
    contrib = torch.full((n,), 7.0, device="cuda")      # poisoned: must be overwritten
    for _ in range(3):
        try:
            ren.render_contrib(sf, c, contrib, **im)
            ren.stats()
            break
        except sgs.SgsError as e:
            if e.status != sgs.SGS_WORKSPACE_OVERFLOW:
                raise
    return contrib, im


def contrib_exposure(sc, camv, cfg, cam):
    up = np.zeros((8, cam.height, cam.width)); up[0] = 1.0       # d/d rgb_k[0] of sum_p I_r(p) = sum_p w_k(p) = C_k
    return oracle.exposure(sc, camv, cfg, up)["rgb"][:, 0]


def check_contrib(C_gpu, C_ref, expo):
    err = np.abs(C_gpu - C_ref)
    bound = 1e-4 * np.abs(C_ref) + 1e-3 + C_EXPO * expo
    assert (err <= bound).all(), (int((err > bound).sum()), float((err / bound).max()))
    assert C_EXPO * expo.sum() <= 0.01 * C_ref.sum()             # the allowance is a small part of what is compared
    assert ((C_ref == 0) <= (C_gpu <= C_EXPO * expo + 1e-3)).all()


@pytest.mark.parametrize("name,view,radix", [("C1", 0, False), ("C2", 0, False), ("C3", 3, False), ("C5", 0, False),
                                             ("C1", 0, True), ("C2", 0, True)])
def test_contribution_matches_oracle(name, view, radix):
    """radix: under SGS_FLAG_RADIX_BINNING the tile lists hold compact visible indices; the contribution must still land
    on the splat itself (it used to land on the list value)."""
    sc, cams, _ = scenegen.make_config(name)
    cam = cams[view]
    camv, cfg = oracle.make_cam(cam), oracle.make_cfg()
    ren = sgs.Renderer(async_mode=(name != "C1"), radix_binning=radix)
    t, sf = to_device(sc)
    contrib, im = gpu_contrib(ren, sf, sc.n, cam)
    C_gpu = contrib.cpu().numpy().astype(np.float64)
    C_ref = oracle.contribution(sc, camv, cfg)
    check_contrib(C_gpu, C_ref, contrib_exposure(sc, camv, cfg, cam))
    culled = oracle.binning(sc, camv, cfg)["culled"].astype(bool)
    assert (C_gpu[culled] == 0).all()                                    # exactly zero for inactive / culled
    # sum_k C_k = sum_p O(p) on the GPU's own outputs (Eq. 21 vs Eq. 8)
    assert abs(C_gpu.sum() - planes(im)[7].sum()) <= 1e-4 * C_gpu.sum()
    # the images are those of sgs_render
    im2 = alloc_images(cam)
    ren.render(sf, camera(cam), **im2)
    assert np.array_equal(planes(im), planes(im2))
    ren.close()


def test_covisibility_counts_are_exact_on_oracle_inputs():
    """The kernel on the ORACLE's contributions (rounded to float32) reproduces the oracle's integer counts."""
    sc, cams, _ = scenegen.make_config("C3", n_override=60000)
    cfg = oracle.make_cfg()
    CA = oracle.contribution(sc, oracle.make_cam(cams[0]), cfg).astype(np.float32)
    CB = oracle.contribution(sc, oracle.make_cam(cams[5]), cfg).astype(np.float32)
    act = (scenegen.SplitMix(77).uniform(sc.n) < 0.7).astype(np.uint8)
    ren = sgs.Renderer()
    a, b = torch.from_numpy(CA).cuda(), torch.from_numpy(CB).cuda()
    res = torch.zeros(3, device="cuda")
    for active in (None, act):
        ren.covisibility(a, b, res, active=None if active is None else torch.from_numpy(active).cuda())
        score, inter, union = oracle.covisibility(CA, CB, active)
        got = res.cpu().numpy()
        assert inter > 100 and union > inter
        assert (int(got[1]), int(got[2])) == (inter, union)
        assert abs(got[0] - score) <= 1e-6
    ren.covisibility(torch.zeros(10, device="cuda"), torch.zeros(10, device="cuda"), res)   # empty union -> 0
    assert res.cpu().numpy().tolist() == [0.0, 0.0, 0.0]
    ren.close()


def test_covisibility_end_to_end():
    """Two views rendered on the GPU -> contributions -> Eq. 22, against the same chain in the oracle; the counts may
    differ only by splats whose C sits within 1e-3 of the 0.5 threshold."""
    sc, cams, _ = scenegen.make_config("C3", n_override=100000)
    cfg = oracle.make_cfg()
    ren = sgs.Renderer()
    t, sf = to_device(sc)
    Cg, Cr = [], []
    for v in (0, 4):
        contrib, _ = gpu_contrib(ren, sf, sc.n, cams[v])
        Cg.append(contrib.clone())
        Cr.append(oracle.contribution(sc, oracle.make_cam(cams[v]), cfg))
    res = torch.zeros(3, device="cuda")
    ren.covisibility(Cg[0], Cg[1], res)
    score, inter, union = oracle.covisibility(Cr[0], Cr[1])
    near = int(((np.abs(Cr[0] - 0.5) < 1e-3) | (np.abs(Cr[1] - 0.5) < 1e-3)).sum())
    got = res.cpu().numpy()
    assert 0.05 < score < 0.999
    assert abs(int(got[1]) - inter) <= near and abs(int(got[2]) - union) <= near
    assert abs(got[0] - score) <= (2 * near + 1) / max(union, 1)
    ren.close()
