"""The command-line harnesses that drive the library (run_configs, ensemble) run end to end on the
GPU and their output agrees with the oracle on a small workload: they only marshal and print."""
import json

import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def orc():
    from oracle import oracle
    oracle.build()
    return oracle


def test_run_configs_config1_matches_oracle(orc, capsys):
    from paper_2305_12161_b200 import inputs, run_configs
    assert run_configs.main(["--configs", "config1_L64", "--radial"]) == 0
    lines = [json.loads(l) for l in capsys.readouterr().out.splitlines() if l.startswith("{")]
    cps = [l for l in lines if not l.get("summary")]
    w = inputs.WORKLOADS["config1_L64"]
    assert [l["sweep"] for l in cps] == w["times"]
    ref = orc.Oracle(w["L"], w["seeds"][0])
    t = 0
    for l in cps:
        ref.sweep(l["sweep"] - t)
        t = l["sweep"]
        want = ref.measure_full()
        N = w["L"] ** 3
        assert l["n_broken_mean"] == float(want["n_broken"])
        assert abs(l["m"] - (2.0 * want["n_up"] - N) / N) < 1e-15
        assert abs(l["ell_mean"] - want["ell"]) <= 1e-12 * abs(want["ell"])
        rad = ref.measure_radial()
        assert abs(l["ell_radial_mean"] - rad["ell"]) <= 1e-9 * abs(rad["ell"])
    s = [l for l in lines if l.get("summary")][0]
    assert s["kernel"] == "resident" and s["sweeps"] == w["sweeps"] and s["gpu_launches"] > 0


def test_ensemble_small(capsys):
    from paper_2305_12161_b200 import ensemble
    assert ensemble.main(["--L", "64", "--replicas", "7", "--sweeps", "40", "--chunk", "3"]) == 0
    line = json.loads(capsys.readouterr().out.strip().splitlines()[-1])
    assert line["replicas"] == 7 and line["ell_nan"] == 0
    assert sum(line["hist_radial"]["counts"]) == 7
    assert 2.0 < line["ell_radial_mean"] < line["ell_axis_mean"] < 8.0
