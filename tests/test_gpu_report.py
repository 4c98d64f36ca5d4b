"""-m gpu: the measurement reports (paper_1312_1789_b200.report) run end to end on reduced N and print valid JSON;
the config-5 twin conserves energy and lands every particle on t_end."""
import json
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _run(*args):
    p = subprocess.run([sys.executable, "-m", "paper_1312_1789_b200.report", *args], capture_output=True, text=True,
                       timeout=500, cwd=ROOT)
    assert p.returncode == 0, p.stderr[-2000:]
    return [json.loads(l) for l in p.stdout.splitlines() if l.startswith("{")]


def test_sweep_config2_reduced():
    out = _run("sweep", "--config", "2", "--n", "8192")
    assert out[0]["call"] == "predict" and out[0]["us"] > 0
    forces = [d for d in out if d["call"] == "force"]
    assert [d["n_act"] for d in forces] == [1, 16, 256, 4096, 8192]
    for d in forces:
        assert d["interactions_per_s"] > 0 and d["geometry"]["i_per_thread"] == 2
    # small blocks use many CTAs (j-split) instead of one
    assert forces[0]["geometry"]["ctas"] >= 32


@pytest.mark.parametrize("order", [6, 8])
def test_integrate_config5_twin(order):
    out = _run("integrate", "--config", "5", "--n", "4096", "--order", str(order), "--dt-max-log2", "8")
    d = out[-1]
    assert d["call"] == "integrate" and d["reached_t_end"] is True and d["time_reached"] == 0.0625
    assert d["dt_criterion_order"] == 4
    assert d["rel_energy_error"] < 1e-7, d["rel_energy_error"]  # mixed-precision floor of a 4096-body twin
    assert d["blocks"] > 100 and d["pairs"] > 0
