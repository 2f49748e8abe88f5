"""sgs_map_correction_static (include/sgs.h): the allocation-free variant of sgs_map_correction, whose per-keyframe scratch is a
static device array, against the existing ctx path.  Both run the same kernels, so the results are compared BIT FOR BIT
(tighter than the 2e-6 / 5e-6 bars of test_gpu_map_correction.py), on two calls in a row: the second with fewer keyframes and
other poses, so that anything the first call left in the shared array would show.  This file sorts last on purpose: the
suite runs with pytest -x."""
import numpy as np
import pytest
import torch

import scenegen

pytestmark = pytest.mark.gpu

sgs = pytest.importorskip("paper_2506_00970_b200")


def poses(g, k, ang):
    from scipy.spatial.transform import Rotation
    rot = Rotation.from_rotvec(ang * np.stack([g.normal(3) for _ in range(k)]))
    T = np.zeros((k, 3, 4), np.float32)
    T[:, :, :3] = rot.as_matrix(); T[:, :, 3] = 3.0 * np.stack([g.normal(3) for _ in range(k)])
    return T


def _case(seed, n, K, ang):
    g = scenegen.SplitMix(seed)
    To, Tn = poses(g, K, 1.0), poses(g, K, ang)
    mean = np.stack([g.normal(n) for _ in range(3)], 1).astype(np.float32) * 3
    quat = (np.stack([g.normal(n) for _ in range(4)], 1) * 1.3).astype(np.float32)
    fid = (g.uniform(n) * (K + 2)).astype(np.int32) - 1          # a few ids are -1 or K: no keyframe
    return mean, quat, fid, To.reshape(K, 12), Tn.reshape(K, 12)


def test_static_map_correction_equals_the_ctx_path_on_two_calls_in_a_row():
    d = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    ren = sgs.Renderer()
    for seed, n, K, ang in ((31, 100003, 37, 1.5), (32, 4099, 5, 3.1)):
        mean, quat, fid, To, Tn = _case(seed, n, K, ang)
        m_ref, q_ref = d(mean), d(quat)
        ren.map_correction(m_ref, q_ref, d(fid), d(To), d(Tn))
        m_st, q_st, f_d, To_d, Tn_d = d(mean), d(quat), d(fid), d(To), d(Tn)     # every buffer exists before the call
        torch.cuda.synchronize()
        before = torch.cuda.memory_allocated()
        sgs.map_correction_static(m_st, q_st, f_d, To_d, Tn_d)
        assert torch.cuda.memory_allocated() == before
        torch.cuda.synchronize()
        assert not torch.equal(m_st.cpu(), torch.from_numpy(mean))            # something was corrected
        assert torch.equal(m_st, m_ref) and torch.equal(q_st, q_ref)
    ren.close()


def test_static_map_correction_rejects_sizes_beyond_its_limit():
    K = sgs.SGS_STATIC_MAX_FRAMES + 1
    m, q = torch.ones(8, 3, device="cuda"), torch.ones(8, 4, device="cuda")
    f = torch.zeros(8, dtype=torch.int32, device="cuda")
    T = torch.zeros(K, 12, device="cuda")
    with pytest.raises(sgs.SgsError) as e:
        sgs.map_correction_static(m, q, f, T, T)
    assert e.value.status == sgs.SGS_LIMIT_EXCEEDED and "SGS_STATIC_MAX_FRAMES" in str(e.value)
    torch.cuda.synchronize()
    assert float(m.min()) == 1.0 and float(q.max()) == 1.0                      # nothing was touched
    Tm = torch.eye(3, 4, device="cuda").reshape(1, 12).repeat(sgs.SGS_STATIC_MAX_FRAMES, 1).contiguous()
    sgs.map_correction_static(m, q, f, Tm, Tm)                                  # exactly the limit: accepted (identity)
    torch.cuda.synchronize()
    assert torch.equal(m, torch.ones(8, 3, device="cuda"))
