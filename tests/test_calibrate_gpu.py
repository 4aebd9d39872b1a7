"""GPU parity of smre_calibrate (threshold calibration, sec. 2.1) against the oracle.

Tolerance: the kernel adds the s^2 positive squares of a window sequentially in fp32, so
|dt| / t <= s^2 u (u = 2^-24); with t ~ s^2 and sigma_s = 1 / (sqrt 8 sqrt s) the statistic moves by at most
t^(1/4) / (4 sigma_s) * s^2 u ~ 0.71 s^3 u.  The quantile is an order statistic: it is compared as the SAME frame's
value (bit-exact selection among the kernel's own Q), the table within the same relative bound.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")
import paper_1503_03492_b200 as smre  # noqa: E402

U = 2.0 ** -24


def q_tol(sides):
    return max(0.71 * max(sides) ** 3 * U, 4e-6)


@pytest.mark.parametrize("n,H,W,sides,alpha", [(40, 64, 64, [1, 2, 3, 4, 5, 6, 7, 8], 0.9),       # the configs' sides
                                               (25, 37, 53, [3, 1, 6], 0.5),                      # ragged, unordered
                                               (12, 70, 45, [1, 2, 4, 8, 16], 0.95),              # C3's ICD levels
                                               (6, 40, 80, [32, 17, 2], 1.0),                     # largest side
                                               (9, 33, 33, [33 - 1], 0.3),                        # one window row / column pair
                                               (300, 16, 16, [1, 2, 4], 0.8)])                    # many small frames
def test_calibration_matches_oracle(oracle, n, H, W, sides, alpha):
    rng = np.random.default_rng(n + H)
    noise = rng.standard_normal((n, H, W)).astype(np.float32)
    noise[0, -1, :] *= 3.0                                       # the last row / column must be seen
    noise[1 % n, :, -1] *= 3.0
    alpha = float(np.float32(alpha))                             # the ABI takes a float: the rank is ceil(alpha_f32 * n)
    c, qa, q = smre.calibrate(torch.from_numpy(noise).cuda(), sides, alpha)
    torch.cuda.synchronize()
    c, qa, q = c.cpu().numpy().astype(np.float64), float(qa.cpu()[0]), q.cpu().numpy().astype(np.float64)
    q_ref = oracle.q_stat(noise, sides)
    tol = q_tol(sides)
    assert np.abs(q - q_ref).max() <= tol, (np.abs(q - q_ref).max(), tol)
    # the quantile: the order statistic of the kernel's own values, and within tol of the oracle's
    k = min(n, max(1, int(np.ceil(alpha * n))))
    assert qa == np.sort(q.astype(np.float32))[k - 1]
    qa_ref, c_ref = oracle.thresholds_from_q(q_ref, alpha, sides)
    assert abs(qa - qa_ref) <= tol
    # thresholds: exact formula on the kernel's quantile (fp32 rounding), and close to the oracle's table
    _, c_from_qa = oracle.thresholds_from_q([qa], 1.0, sides)
    np.testing.assert_allclose(c, c_from_qa, rtol=2e-6)
    np.testing.assert_allclose(c, c_ref, rtol=2e-6 + 4 * tol)
    # deterministic
    c2, qa2, q2 = smre.calibrate(torch.from_numpy(noise).cuda(), sides, alpha)
    assert torch.equal(q2.cpu(), torch.from_numpy(q.astype(np.float32))) and float(qa2.cpu()[0]) == qa


def test_calibrated_table_drives_the_projection(oracle):
    """The table smre_calibrate writes is the table smre_create takes: project a noisy image with it, against the
    oracle run with the same table."""
    import smre_inputs as si
    from tests import parity
    rng = np.random.default_rng(77)
    sides = [1, 2, 3, 4]
    noise = torch.from_numpy(rng.standard_normal((200, 48, 48)).astype(np.float32)).cuda()
    c, qa, q = smre.calibrate(noise, sides, 0.9)
    c = c.cpu().numpy()
    w = si.config(0)
    sol = smre.Solver(w.H, w.W, sides, c, "standard")
    x = sol.project(torch.from_numpy(w.y).cuda(), 20)
    torch.cuda.synchronize()
    d = parity.compare(oracle, w.y, x.cpu().numpy(), oracle.project(w.y, sides, c, 20, "standard"), sides, c, "standard")
    assert np.abs(x.cpu().numpy() - w.y).max() > 0.05 and d["max_abs_err"] < 2e-5
    sol.close()


def test_calibrate_errors():
    z = torch.zeros(2, 8, 8, device="cuda")
    out = torch.zeros(8, device="cuda")
    for sides, alpha in (([9], 0.5), ([2, 2], 0.5), ([1], 0.0), ([1], 1.5), ([0], 0.5)):
        with pytest.raises(smre.SmreError) as e:
            smre.smre_calibrate(8, 8, 2, sides, z.data_ptr(), alpha, out.data_ptr(), out.data_ptr(), out.data_ptr())
        assert e.value.status == smre.smre.SMRE_EINVAL
    with pytest.raises(smre.SmreError):
        smre.smre_calibrate(8, 8, 2, [1], None, 0.5, out.data_ptr(), out.data_ptr(), out.data_ptr())


@pytest.mark.parametrize("n,H,W", [(64, 256, 256), (7, 33, 35), (2, 5, 4), (1, 16, 16)])
def test_cumulant2_matches_oracle(oracle, n, H, W):
    """Eq. 19 on a SOFI-like stack: bright background, blinking emitters."""
    rng = np.random.default_rng(n + W)
    stack = (200.0 + 3.0 * rng.standard_normal((n, H, W))).astype(np.float32)
    stack[:, H // 2, W // 2] += (40.0 * (rng.random(n) < 0.5)).astype(np.float32)      # a blinking emitter
    c2 = smre.cumulant2(torch.from_numpy(stack).cuda())
    torch.cuda.synchronize()
    ref = oracle.cumulant2(stack)
    # fp32 moments about the first frame: deviations ~ 10, n terms -> relative 1e-5 of the variance scale is ample
    assert np.abs(c2.cpu().numpy() - ref).max() <= 2e-5 * max(1.0, float(ref.max()))
    if n > 1:
        assert ref[H // 2, W // 2] > 5 * np.median(ref) or n < 4
