"""bench.py's JSON line (`-m gpu`): the contract keys of the task, on a small population so that it runs in seconds."""
import json
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    return torch


@pytest.fixture(scope="module")
def sc():
    import paper_2408_13170_b200 as sc
    sc.load_library()          # fails loudly if the extension is missing
    return sc


def test_bench_line_has_the_contract_keys():
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--particles", "512", "--steps", "2", "--warmup", "3",
                          "--no-cpu-baseline"], capture_output=True, text=True, timeout=600)
    assert out.returncode == 0, out.stderr[-2000:]
    line = json.loads(out.stdout.strip().splitlines()[-1])
    for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling", "vs_baseline",
              "dtype", "data", "config", "roofline", "e2e", "gpu_launches", "clocks"):
        assert k in line, k
    assert line["n_gpus"] == 1 and line["steps"] == 2 and line["warmup"] == 3 and line["higher_is_better"] is True
    assert "workload" in line["config"] and line["config"]["workload"].startswith("c3")
    assert line["value"] > 0 and line["gpu_launches"] > 0 and line["vs_baseline"] is None
    # value counts evaluated (particle, bin) pairs: never more than the nominal rate
    assert line["value"] <= line["nominal_particle_bin_per_s"] * (1 + 1e-12) and 0 < line["evaluated_fraction"] <= 1
    r = line["roofline"]
    for k in ("bound", "achieved", "peak", "unit", "frac", "traffic", "frac_pipe_fma", "frac_model"):
        assert k in r, k
    assert r["bound"] == "alu" and r["unit"] == "TFLOP/s" and 0 < r["frac"] < 1 and r["frac"] == r["frac_pipe_fma"]
    assert r["frac"] == pytest.approx(r["achieved"] / r["peak"], rel=1e-9)
    e = line["e2e"]
    assert e["value"] > 0 and e["h2d_bytes_per_step"] == 512 * 72 and e["d2h_bytes_per_step"] == 512 * 72
    for k in ("adaptive_segments_N100", "coherent_N1", "tensor_core_flavour", "three_channels", "streams_x_one_template"):
        assert k in line["extras"], k
    assert "ms_per_eval" in line["extras"]["three_channels"] and "ms_per_eval" in line["extras"]["coherent_N1"]


def test_launch_info_and_window_fraction_hint(torch_cuda, sc):
    """sc_get_launch_info reports the node spacing and flavour of the last FP32-amplitude pass; stating the window fraction
    (SC_OPT_WINDOW_FRACTION_PPM) widens the spacing with the number of segments per particle and never touches per-segment output."""
    import numpy as np
    import sc_synth as sy
    inp = sy.config_inputs(3, P=256)
    t = lambda a: torch_cuda.from_numpy(np.ascontiguousarray(a)).to("cuda:0")
    H = sc.Handle(inp["cfg"], torch_cuda.view_as_real(t(inp["noise_A"])).contiguous(), torch_cuda.view_as_real(t(inp["noise_E"])).contiguous(),
                  t(inp["S_A"]), t(inp["S_E"]))
    assert H.launch_info() == (0, 0)
    H.set_option(sc.SC_OPT_TC_MAX_S, int(np.ceil(inp["hi"][2])))
    par, e = t(inp["particles"]), inp["edges"][5000]
    a = H.eval_stat(par, e).cpu().numpy()
    lg0, fl0 = H.launch_info()
    assert lg0 == 10 and fl0 & sc.SC_FLAVOUR_MUFU and fl0 & sc.SC_FLAVOUR_MERGE
    phi = H.counters()[0] / (256 * inp["cfg"]["n_bins"])
    H.set_option(sc.SC_OPT_WINDOW_FRACTION_PPM, int(round(1e6 * phi)))
    b = H.eval_stat(par, e).cpu().numpy()
    lg1, fl1 = H.launch_info()
    assert lg1 == 11 and fl1 & sc.SC_FLAVOUR_QUAD              # N' ~ 2500 segments per particle: 4 (N'/8)^(1/12) = 6.5 days >= 4.4
    live = a > 0
    assert np.all(np.abs(b[live] - a[live]) <= 1e-7 * a[live])
    H.eval_stat(par, sy.edges(inp["cfg"]["n_bins"], 8))        # N' = 4: the spacing of N' = 8
    assert H.launch_info()[0] == 10
    H.eval_segments(par, e)                                    # per-segment output: nothing averages
    assert H.launch_info()[0] == 10
    with pytest.raises(sc.SCError):
        H.set_option(sc.SC_OPT_WINDOW_FRACTION_PPM, 1000001)
    H.close()


def test_quadratic_amplitude_runs_are_a_small_perturbation(torch_cuda, sc):
    """SC_OPT_QUAD_AMPLITUDES: the QUAD flavour of the pair loop (shared edges and per-particle segments) against the cubic one on
    the same handle -- the economised u^3 term is <= 3e-8 of the amplitude, so Upsilon moves by far less than the 1e-6 bar."""
    import numpy as np
    import sc_synth as sy
    inp = sy.config_inputs(3, P=512)
    t = lambda a: torch_cuda.from_numpy(np.ascontiguousarray(a)).to("cuda:0")
    H = sc.Handle(inp["cfg"], torch_cuda.view_as_real(t(inp["noise_A"])).contiguous(), torch_cuda.view_as_real(t(inp["noise_E"])).contiguous(),
                  t(inp["S_A"]), t(inp["S_E"]))
    H.set_option(sc.SC_OPT_TC_MAX_S, int(np.ceil(inp["hi"][2])))
    par, e = t(inp["particles"]), inp["edges"][5000]
    st = torch_cuda.empty(512, dtype=torch_cuda.float64, device="cuda:0")
    out = {}
    for quad in (1, 0):
        H.set_option(sc.SC_OPT_QUAD_AMPLITUDES, quad)
        out[("shared", quad)] = H.eval_stat(par, e).cpu().numpy()
        assert bool(H.launch_info()[1] & sc.SC_FLAVOUR_QUAD) == bool(quad)
        sc.sc_eval_stat_adaptive(H.h, par, 512, 100, st)
        out[("adaptive", quad)] = st.cpu().numpy().copy()
    for kind in ("shared", "adaptive"):
        a, b = out[(kind, 1)], out[(kind, 0)]
        live = b > 0
        d = np.abs(a[live] - b[live]) / b[live]
        assert live.sum() > 400 and d.max() < 5e-8 and d.max() > 0, (kind, d.max())
    H.close()
