"""The reciprocal routines the kernels use instead of IEEE sqrt and divide (common.cuh: rsqrt_fast, rinv3_fast,
rcp_fast, built on the MUFU.RSQ64H / MUFU.RCP64H seeds).  The paper keeps IEEE operations because an rsqrt with a
BIASED error would accumulate over millions of steps.  Here the signed error of each routine is
measured in ulps over 1e8 log-uniform inputs against a reference carried in extended precision (x87 long double, 64-bit
mantissa: 11 bits more than FP64), and the test asserts that the mean signed error is zero to 0.01 ulp and the
maximum stays at a few ulps."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

N_TOTAL = 100_000_000
CHUNK = 5_000_000


@pytest.mark.skipif(np.finfo(np.longdouble).nmant < 63, reason="needs an 80-bit long double for the reference")
@pytest.mark.parametrize("which,name,power,max_ulp", [(0, "rsqrt_fast", -0.5, 1.6), (1, "rinv3_fast", -1.5, 4.5), (2, "rcp_fast", -1.0, 1.1)])
def test_reciprocal_routines_are_unbiased(which, name, power, max_ulp):
    import torch
    import paper_1404_2324_b200 as G
    from paper_1404_2324_b200 import build
    build.build()
    g = G.Genga(0, 4)
    rng = np.random.default_rng(1234 + which)
    ld = np.longdouble
    tot, worst, n = ld(0), 0.0, 0
    for _ in range(N_TOTAL // CHUNK):
        # log-uniform over 1e-12 .. 1e12 (squared distances in AU^2 from 1e-6 AU to 1e6 AU), random mantissas
        x = 10.0 ** rng.uniform(-12.0, 12.0, CHUNK)
        y = g.eval_fast(which, torch.from_numpy(x).cuda()).cpu().numpy()
        xl, yl = x.astype(ld), y.astype(ld)
        # relative error of y against x^power without forming the reference by a rounded operation:
        #   x^-1/2: x y^2 - 1 = 2 d;   x^-3/2: x^3 y^2 - 1 = 2 d;   1/x: x y - 1 = d      (d = relative error, |d| << 1)
        if which == 0:
            d = (xl * yl * yl - 1) / 2
        elif which == 1:
            d = (xl * xl * xl * yl * yl - 1) / 2
        else:
            d = xl * yl - 1
        ulp = np.spacing(np.abs(y)).astype(ld) / yl           # one ulp of y, relative
        e = d / ulp
        tot += e.sum()
        worst = max(worst, float(np.abs(e).max()))
        n += CHUNK
    mean = float(tot / n)
    print("%s: mean signed error %+.5f ulp, max |error| %.3f ulp over %d samples" % (name, mean, worst, n))
    assert abs(mean) < 0.01, (name, mean)
    assert worst < max_ulp, (name, worst)
    g.close()
