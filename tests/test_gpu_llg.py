"""NEXT row 4: the minimal LLG RK4 integrator that consumes the convolution, with the sub-step
extrapolation of the demagnetizing field, judged with the error metric of PAPER.md:47
(eps = sum_i ||M(t_i) - M~(t_i)|| / (n Ms) over the recorded mesh-averaged magnetisation; the paper's fp32 floor is
~1e-4).  The reference trajectories are the oracle's (fp64 NumPy RK4 on Eq. (5), H_d by the FFT cross-check of Eq. (1))."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

EPS_FP32 = 1e-4          # "the lower precision limits the accuracy ... which is ~1e-4"


@pytest.fixture(scope="module")
def torch():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    return torch


@pytest.fixture(scope="module")
def B():
    from paper_2308_08447_b200 import binding
    binding.lib()
    return binding


def film_state(n, Ms, seed):
    """Film magnetised mostly along +x with a seeded random tilt: the switching field of PAPER.md:47 then reverses it."""
    from paper_2308_08447_b200 import workloads as W
    M = W.random_unit_vectors(n, Ms, seed).astype(np.float64)
    M[0] += 2.0 * Ms
    M *= Ms / np.sqrt((M * M).sum(axis=0, keepdims=True))
    return M.astype(np.float32)


def run_gpu(torch, B, n, h, Ms, M0, Hz, alpha, dt, steps, prec, extrapolate, T=None):
    dtp = torch.float32 if prec == 0 else torch.float64
    with B.Plan(n, h, 0, prec) as p:
        p.set_kernel(T)
        with B.LLG(p, Ms, alpha) as L:
            L.set_field(Hz)
            M = torch.from_numpy(M0).to("cuda", dtp)
            rec = torch.zeros((steps + 1, 3), dtype=torch.float64, device="cuda")
            L.mean(M, rec[0])
            for i in range(steps):
                L.step(M, dt, extrapolate)
                L.mean(M, rec[i + 1])
            torch.cuda.synchronize()
            return M.cpu().numpy().astype(np.float64), rec.cpu().numpy(), L.counts()


@pytest.mark.parametrize("prec", [0, 1])
def test_llg_trajectory_matches_the_oracle(torch, B, oracle, prec):
    """64 x 32 x 2 film of 5 nm cells (the cell size and Ms of PAPER.md:47), switching field (-20, 1, 0) kA/m,
    200 RK4 steps of 100 fs, the demagnetizing field convolved at every stage on both sides."""
    n, h, Ms = (64, 32, 2), (5e-9, 5e-9, 5e-9), 8e5
    Hz, alpha, dt, steps = (-2.0e4, 1.0e3, 0.0), 0.1, 1.0e-13, 200
    M0 = film_state(n, Ms, 7)
    Tn = oracle.tensor_table(n, h)
    Mref, avg_ref, nc_ref = oracle.llg_rk4_run(Tn, M0.astype(np.float64), Ms, Hz, alpha, dt, steps)
    Mg, avg, cnt = run_gpu(torch, B, n, h, Ms, M0, Hz, alpha, dt, steps, prec, False, T=Tn)
    eps = oracle.fig2_error(avg, avg_ref, Ms)
    assert cnt["convolutions"] == nc_ref == 4 * steps and cnt["extrapolations"] == 0
    assert abs(cnt["time"] - steps * dt) < 1e-20
    assert eps <= (EPS_FP32 if prec == 0 else 1e-10), eps
    assert np.abs(Mg - Mref).max() / Ms <= (2e-4 if prec == 0 else 1e-9)
    norm0 = np.sqrt((M0.astype(np.float64) ** 2).sum(axis=0))              # fp32-rounded unit vectors: |M0| = Ms (1 +- 6e-8)
    assert np.abs(np.sqrt((Mg * Mg).sum(axis=0)) / norm0 - 1.0).max() <= (1e-4 if prec == 0 else 1e-9)  # |M| kept
    assert np.abs(avg_ref[-1] - avg_ref[0]).max() / Ms > 1e-3                                         # something moved


def test_llg_with_extrapolated_substep_fields(torch, B, oracle, capsys):
    """the run whose sub-step fields are the quartic through the five last computed fields must stay within
    the paper's error floor of (i) the GPU run that convolves at every stage and (ii) the oracle's run of the same
    scheme, while enqueuing at most half the convolutions (here 16 + (steps - 4) instead of 4 steps)."""
    n, h, Ms = (64, 32, 2), (5e-9, 5e-9, 5e-9), 8e5
    Hz, alpha, dt, steps = (-2.0e4, 1.0e3, 0.0), 0.1, 1.0e-13, 200
    M0 = film_state(n, Ms, 7)
    Tn = oracle.tensor_table(n, h)
    Mf, avg_full, cf = run_gpu(torch, B, n, h, Ms, M0, Hz, alpha, dt, steps, 0, False, T=Tn)
    Mx, avg_ext, cx = run_gpu(torch, B, n, h, Ms, M0, Hz, alpha, dt, steps, 0, True, T=Tn)
    _, avg_oext, nc_oext = oracle.llg_rk4_run(Tn, M0.astype(np.float64), Ms, Hz, alpha, dt, steps, extrapolate=True)
    assert cf["convolutions"] == 4 * steps
    assert cx["convolutions"] == nc_oext == 16 + (steps - 4)
    assert cx["extrapolations"] == 2 * (steps - 4)                      # t + dt/2 (shared by stages 2 and 3) and t + dt
    assert 2 * cx["convolutions"] <= cf["convolutions"]
    e_gpu = oracle.fig2_error(avg_ext, avg_full, Ms)
    e_orc = oracle.fig2_error(avg_ext, avg_oext, Ms)
    assert e_gpu <= EPS_FP32 and e_orc <= EPS_FP32, (e_gpu, e_orc)
    with capsys.disabled():
        print(f"\n[llg] {steps} RK4 steps: {cf['convolutions']} convolutions without extrapolation, {cx['convolutions']} + "
              f"{cx['extrapolations']} extrapolation passes with it ({cx['convolutions'] / cf['convolutions']:.3f} of the "
              f"convolutions); eps vs every-stage run {e_gpu:.2e}, vs oracle {e_orc:.2e}")


def test_llg_built_in_tensor_embedded_mesh_and_errors(torch, B, oracle):
    """The integrator goes through the public calls, so it works on a general (embedded) mesh with the built-in tensor;
    bad arguments are rejected."""
    n, h, Ms = (24, 10, 3), (4e-9, 5e-9, 3e-9), 8e5
    Hz, alpha, dt, steps = (1.0e4, -3.0e4, 5.0e3), 0.05, 5.0e-14, 40
    M0 = film_state(n, Ms, 9)
    Tn = oracle.tensor_table(n, h)
    _, avg_ref, _ = oracle.llg_rk4_run(Tn, M0.astype(np.float64), Ms, Hz, alpha, dt, steps, extrapolate=True)
    _, avg, cnt = run_gpu(torch, B, n, h, Ms, M0, Hz, alpha, dt, steps, 0, True, T=None)
    assert oracle.fig2_error(avg, avg_ref, Ms) <= EPS_FP32
    with B.Plan(n, h, 0, 0) as p:
        p.set_kernel(None)
        for bad in ((0.0, 0.1), (8e5, -1.0), (float("nan"), 0.1)):
            with pytest.raises(B.DemagError) as e:
                B.LLG(p, bad[0], bad[1])
            assert e.value.status == 1
        with B.LLG(p, Ms, alpha) as L:
            M = torch.from_numpy(M0).cuda()
            for dtb in (0.0, -1e-13, float("inf")):
                with pytest.raises(B.DemagError) as e:
                    L.step(M, dtb)
                assert e.value.status == 1
            L.step(M, dt); L.reset()
            assert L.counts() == {"convolutions": 0, "extrapolations": 0, "time": 0.0}
    with B.Plan(n, h, 0, 0) as p:                                         # no kernel yet: the convolution's own error comes through
        with B.LLG(p, Ms, alpha) as L:
            with pytest.raises(B.DemagError) as e:
                L.step(torch.from_numpy(M0).cuda(), dt)
            assert e.value.status == 5
