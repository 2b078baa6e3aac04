"""Row F3: the synthetic injection-recovery workload run
through the CUDA path and, on the same stars, through the fp64 oracle: the depth errors must
agree, and the ordering the paper reports at 1000 ppm (aggressive < default < symmetric,
Tables 1-2) must hold on the generator stars."""
import numpy as np
import pytest

from oracle import umi_oracle as orc
from workloads import injection_recovery as ir
from workloads import lightcurves as lc

pytestmark = pytest.mark.gpu


def test_injection_recovery_gpu_equals_oracle_and_paper_ordering():
    import torch
    import paper_2604_06602_b200 as umi
    umi.lib()
    cfg, flux = lc.make(2, 24)
    depths = (100.0, 1000.0)
    got, ref = {}, {}
    for name, kw in ir.SETTINGS.items():
        def gpu(x, kw=kw):
            _, _, flat = umi.umi_detrend_family(None, torch.from_numpy(x).cuda(), cfg.W, n_iter=cfg.n_iter,
                                                flat=True, **kw)
            return flat.cpu().numpy()

        def cpu(x, kw=kw):
            r = orc.family(x, cfg.W, n_iter=cfg.n_iter, **kw)
            return orc.normalize(x, r.trend64)
        got[name] = ir.depth_errors(flux, cfg.dt_days, gpu, depths)
        ref[name] = ir.depth_errors(flux, cfg.dt_days, cpu, depths)
        # fp32 trend (1e-5 relative bar) vs fp64 trend: depths of 1e-4 .. 1e-3 recovered from
        # ~800 in-transit cadences agree to well under a percentage point
        np.testing.assert_allclose(got[name], ref[name], atol=0.2)
    d, a, s = (got[k][1] for k in list(ir.SETTINGS)[:3])
    assert a < d < s, (a, d, s)
