"""the paper's quality metric (CNR, Eq. (1)) on the GPU against the oracle, and the
paper's own simulation workload (Fig. 1) through the C ABI: the source modulated at the examined
frequency stands out, an "incorrect" frequency shows nothing, fewer frames give less contrast
(PAPER.md:41)."""
import numpy as np
import pytest

from _parity import check_float_maps, oracle_maps

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def Q():
    import torch
    assert torch.cuda.is_available()
    from paper_1511_03390_b200 import qld
    qld.load_library()
    return qld


@pytest.mark.parametrize("H,W,y0,x0,m", [(14, 16, 5, 6, 4), (3, 3, 1, 1, 1), (480, 640, 200, 300, 37), (1024, 1280, 100, 100, 100),
                                         (64, 64, 21, 22, 21)])
def test_cnr_matches_oracle(Q, oracle, H, W, y0, x0, m):
    import torch
    rng = np.random.default_rng(H + m)
    img = rng.normal(1000.0, 30.0, size=(H, W)).astype(np.float32)
    img[y0:y0 + m, x0:x0 + m] += 75.0
    got = Q.cnr(torch.from_numpy(img).cuda(), y0, x0, m).cpu().numpy()
    exp = np.array(oracle.cnr(img, y0, x0, m))
    assert np.allclose(got, exp, rtol=1e-11, atol=0.0), (got, exp)


def test_cnr_degenerate_and_errors(Q, oracle):
    import torch
    flat = torch.zeros((12, 12), dtype=torch.float32, device="cuda")
    assert np.isnan(Q.cnr(flat, 4, 4, 4).cpu().numpy()[0])                    # 0 / 0, as the oracle
    flat[4:8, 4:8] = 2.0
    got = Q.cnr(flat, 4, 4, 4).cpu().numpy()
    assert got[0] == np.inf and tuple(got[1:]) == (2.0, 0.0, 0.0)
    for bad in ((3, 4, 4), (4, 5, 4), (4, 4, 0)):                                # the slice leaves the frame / m < 1
        with pytest.raises(Q.QLDError) as e:
            Q.cnr(flat, *bad)
        assert e.value.status == Q.QLD_E_INVAL


def test_paper_simulation_workload(Q, oracle):
    from paper_1511_03390_b200 import synth
    ps = synth.paper_sim()                              # 96 x 96, m = 8, N = 82, X = 5, 20/23/26/29 Hz at 100 frames/s
    N, n = ps.frames.shape[0], ps.frames.shape[1]

    def run(frames, nu):
        ref = {"nu": nu}
        ctx = Q.QLD(n, n, "u16", frames.shape[0], [ref], accum=Q.QLD_ACC_FP32, maps=Q.QLD_MAP_AMP | Q.QLD_MAP_I | Q.QLD_MAP_Q)
        ctx.push_frames(frames)
        ctx.demod(Q.QLD_WHOLE)
        ctx.sync()
        I, Qm, A, _ = ctx.get_maps(0)
        check_float_maps((I.cpu().numpy(), Qm.cpu().numpy(), A.cpu().numpy(), None), oracle_maps(oracle, frames, ref), what=f"paper sim nu={nu}")
        out = []
        for (y0, x0) in ps.boxes:
            g = Q.cnr(A, y0, x0, ps.m).cpu().numpy()
            o = np.array(oracle.cnr(A.cpu().numpy(), y0, x0, ps.m))                # the oracle's CNR of the same map
            assert np.allclose(g, o, rtol=1e-11), (g, o)
            out.append(float(g[0]))
        ctx.destroy()
        return out

    right = run(ps.frames, ps.nus[1])                   # the "frequency of interest", 23 Hz
    wrong = run(ps.frames, 0.31)                        # the "incorrect" frequency, 31 Hz
    half = run(ps.frames[:N // 2], ps.nus[1])           # N / 2 frames
    assert right[1] > 3.0 and all(abs(c) < 1.0 for i, c in enumerate(right) if i != 1)    # only source 2 is revealed
    assert all(abs(c) < 1.0 for c in wrong)                                               # nothing at the wrong frequency
    assert 1.0 < half[1] < right[1]                                                       # fewer frames, less contrast
