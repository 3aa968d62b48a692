"""Where the oracle itself is not determined to the stated tolerances: a CPU-only demonstration.

Late in config 3 (the robot has left the landmark box, dead-reckons with metre-level uncertainty and re-observes a
landmark) the two-iteration Gauss-Newton recursion with its relinearised marginalisation prior is unstable in a few
environments: ONE float32 ulp in ONE input moves the oracle's own outputs by a large part of a tolerance, and a
1e-13 change of one state variable fifteen steps earlier moves the newest pose by a whole tolerance.  No second
implementation -- fp32 or fp64 -- can be held to 1e-3 there; everywhere else the same changes move the outputs by
1e-6 of a tolerance.  Environment 15740 of config 3 is such a case; the parity tests find these env-steps with
tests/helpers.determined (from the oracle alone) and require that they are at most 1e-3 of all env-steps."""
import numpy as np

import oracle
from harness import synth
from tests.gpu_driver import parity_errors
from tests.helpers import determined, drive


def test_one_input_ulp_moves_the_oracle_where_gn_is_unstable():
    cfg = synth.CONFIGS[3]
    envs = np.array([0, 4096, 8192, 15740], np.int32)
    data = synth.generate(cfg, env_ids=envs)
    ref = oracle.run_batch(data, cfg.iters)
    pd = dict(data)
    od = data["odom"].copy()
    od[0, 0] = np.nextafter(od[0, 0], np.float32(np.inf))
    pd["odom"] = od
    alt = oracle.run_batch(pd, cfg.iters)
    err = parity_errors(dict(poses=alt["poses"], cov=alt["cov"], logdet=alt["logdet"]), ref)
    G = np.max([err[k] for k in err], axis=0)             # in units of the stated tolerances
    assert G[:, :3].max() < 1e-3                          # ordinary environments: far below a tolerance, all 300 steps
    assert G[:290, 3].max() < 1e-3                        # the unstable one: fine for 290 steps ...
    assert G[298:, 3].max() > 0.2                         # ... then its own answer moves by a good part of a tolerance
    det = determined(oracle, data, cfg.iters, None, ref)
    assert det[:, :3].all() and det[:290, 3].all() and not det[299, 3]


def test_state_perturbation_is_amplified_ten_orders_of_magnitude():
    cfg = synth.CONFIGS[3]
    one = synth.generate(cfg, env_ids=np.array([15740], np.int32))

    def run(eps):
        out = []

        def cb(rec, orc):
            out.append(rec["poses"].copy())
            if rec["t"] == 285 and eps:
                v = orc.state()
                v[3] += eps
                orc.set_state(v)
        drive(oracle.Oracle(cfg.W, cfg.L), one, 0, cfg.iters, on_step=cb)
        return out

    a, b = run(0.0), run(1e-13)
    assert np.abs(a[289] - b[289]).max() < 1e-12          # five steps later: still nothing
    assert np.abs(a[299] - b[299]).max() > 1e-4           # fifteen steps later: > 1e-4 m, ~ the pose tolerance at 12 m
