"""Why BASELINE.json configs[3] (two streams in a strong field, dt = 50, ~590 sub-steps per
orbit) cannot meet north_star's fp32 bar of 1e-5 on v per particle while configs[2] does
(DESIGN.md 2 "cfg3 in fp32"): the method itself, run in fp64 by the oracle, amplifies ONE fp32
rounding error of the input velocity by an order of magnitude in cfg3 and damps it in cfg2.  An
fp32 kernel rounds at every sub-step, so its distance from the oracle is about
response x sqrt(n_sub): ~3e-5 for cfg3 (measured on the GPU: 7e-5), ~5e-7 for cfg2 (measured 3e-7).
CPU only: both runs are the oracle's."""
import numpy as np

from paper_1111_5295_b200 import workloads as W
from helpers import ulp_response


def test_one_ulp_response_cfg3_vs_cfg2(oracle):
    r3 = ulp_response(oracle, W.config3(n=20_011))
    r2 = ulp_response(oracle, W.config2(n=50_003))
    eps = 2.0 ** -24                      # rms-ish size of one fp32 rounding, relative
    print(f"[sensitivity] cfg3: {r3}\n[sensitivity] cfg2: {r2}")
    # cfg3 amplifies, cfg2 does not
    assert r3["v"] > 10 * eps and r2["v"] < 2 * eps
    assert r3["n_sub_mean"] > 500 and r2["n_sub_mean"] < 60
    # the random-walk estimate of an fp32 kernel's error: above the 1e-5 bar for cfg3, far below
    # it for cfg2
    est3, est2 = r3["v"] * np.sqrt(r3["n_sub_mean"]), r2["v"] * np.sqrt(r2["n_sub_mean"])
    assert est3 > 1e-5 and est2 < 1e-6
