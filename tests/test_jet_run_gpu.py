"""The long-run driver (paper_2403_15773_b200/jet_run.py) on a small jet: runs through the C-ABI,
keeps the fields physical, samples the mid-plane averages and reports the paper's diagnostics."""
import json
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("forcing", ["kick", "guo"])
def test_jet_run_small(tmp_path, forcing):
    out = tmp_path / "jet.json"
    cmd = [sys.executable, "-m", "paper_2403_15773_b200.jet_run", "--grid", "64", "64", "160", "--D", "8",
           "--We", "200", "--Re", "500", "--steps", "1600", "--avg-from", "800", "--chunk", "400", "--every", "4",
           "--forcing", forcing, "--out", str(out)]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stderr[-2000:]
    d = json.loads(out.read_text())
    assert d["blew_up_at_step"] is None and d["steps_done"] == 1600 and d["nsamples"] == 200
    assert ("guo" in d["kernel"]) == (forcing == "guo")
    assert -0.05 < d["phi_range"][0] and d["phi_range"][1] < 1.05
    assert 0.95 < d["rho_range"][0] and d["rho_range"][1] < 1.05
    # the jet core: centre-line phi and velocity near the nozzle stay at their inlet values
    assert d["phi_c"][0] > 0.99 and abs(d["uc_over_U"][0] - 1.0) < 0.06
    assert d["uc_over_U"][-1] < 0.5          # and the jet has not reached the outlet at full speed
