"""One molecular-dynamics trajectory of a BASELINE config on the GPU, with per-step observables.

    python -m paper_1212_0785_b200.trajectory --config 5 --dtype f64 [--nsteps 20] [--no-observables]

Momentum refresh and hot start from the counter-based generator, then ONE library call:
`qcd_trajectory` (leapfrog of single-pass steps, PAPER.md:17 operations, integrator R6) returns the plaquette,
the per-timeslice plaquette and the kinetic energy of every step as by-products of the force kernel (no extra
pass over the fields), hence H before, H after and dH.  `--no-observables` runs `qcd_leapfrog_single_pass`.
Prints one JSON line: site-updates/s over the trajectory (CUDA events), the HBM fraction the step's algorithmic
bytes correspond to, plaquette / K / H before and after, dH, and the per-step (plaquette, K) series.
BASELINE.json config 5 ("sustained 20-step leapfrog trajectory with per-step reunitarization and reductions")
is `--config 5`.
"""
import argparse
import json
import os
import sys

import torch

from . import binding as qcd

SEED_BASE = 0x1212078500000000
CONFIGS = {
    1: dict(dims=(4, 4, 4, 4), sigma=0.5, beta=5.6, eps=0.1, nsteps=1),
    2: dict(dims=(8, 8, 8, 16), sigma=0.5, beta=5.8, eps=0.05, nsteps=10),
    3: dict(dims=(16, 16, 16, 32), sigma=0.5, beta=5.8, eps=0.05, nsteps=10),
    4: dict(dims=(32, 32, 32, 64), sigma=0.2, beta=6.0, eps=0.02, nsteps=20),
    5: dict(dims=(48, 48, 48, 96), sigma=0.3, beta=6.2, eps=0.01, nsteps=20),
}


def run(config, dtype=torch.float64, nsteps=None, observables=True):
    c = CONFIGS[config]
    dims, beta, eps = c["dims"], c["beta"], c["eps"]
    n = nsteps or c["nsteps"]
    seed = SEED_BASE + config
    lat = qcd.Lattice(dims)
    V, Lt = lat.V, dims[3]
    U, P, W = lat.new_matrix_field(dtype), lat.new_matrix_field(dtype), lat.new_matrix_field(dtype)
    ws = lat.new_workspace()
    qcd.qcd_hot_start(lat, U, seed, c["sigma"])
    qcd.qcd_mom_refresh(lat, P, seed)
    obs = torch.zeros((n + 1, 2), dtype=torch.float64, device="cuda")
    per_t = torch.zeros((n + 1, Lt), dtype=torch.float64, device="cuda")
    stream = torch.cuda.current_stream()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record(stream)
    if observables:  # one library call: the integrator and every reduction run inside libqcdmd (qcd_trajectory)
        qcd.qcd_trajectory(lat, U, P, W, beta, eps, n, obs, per_t, ws)
    else:
        qcd.qcd_leapfrog_single_pass(lat, U, P, W, beta, eps, n)
    e1.record(stream)
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1)
    end = torch.zeros(2, dtype=torch.float64, device="cuda")  # stand-alone reductions at the end
    qcd.qcd_plaquette(lat, U, end[0:1], None, ws)
    qcd.qcd_sum(lat, qcd.SUM_NORM2, 72, P, end[1:2], ws)
    o, e = obs.cpu().numpy(), end.cpu().numpy()

    def H(plaq, K):
        return float(K + beta * 6 * V * (1 - plaq))

    rb = 8 if dtype == torch.float64 else 4
    peak = 6532.5
    pk = os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "MEASURED_PEAKS.json")
    if os.path.exists(pk):
        peak = float(json.load(open(pk))["hbm_gbs"])
    gbs = 288 * rb * V * n / (ms * 1e-3) / 1e9  # single-pass steps: 288 reals per site and step
    line = {"config": config, "dims": list(dims), "dtype": "f64" if rb == 8 else "f32", "nsteps": n, "eps": eps,
            "beta": beta, "observables_every_step": observables, "ms": ms, "ms_per_step": ms / n,
            "site_updates_per_s": V * n / (ms * 1e-3), "step_hbm_gbs": gbs, "step_frac_of_hbm_peak": gbs / peak,
            "plaq_end": float(e[0]), "K_end": float(e[1]), "H_end": H(e[0], e[1])}
    if observables:
        line.update({"plaq_start": float(o[0, 0]), "K_start": float(o[0, 1]), "H_start": H(*o[0]),
                     "dH": H(*o[n]) - H(*o[0]), "H_end_from_fused_sums": H(*o[n]),
                     "K_per_16V_start": float(o[0, 1] / (16 * V)),
                     "per_step_plaq_K": [[float(a), float(b)] for a, b in o],
                     "plaq_per_timeslice_end": [float(x) for x in per_t[n].cpu().numpy()]})
    return line


def main(argv=None):
    ap = argparse.ArgumentParser(description=__doc__.split("\n\n")[0])
    ap.add_argument("--config", type=int, default=5, choices=sorted(CONFIGS))
    ap.add_argument("--dtype", default="f64", choices=["f64", "f32"])
    ap.add_argument("--nsteps", type=int, default=None)
    ap.add_argument("--no-observables", action="store_true")
    a = ap.parse_args(argv)
    if not torch.cuda.is_available():
        raise SystemExit("trajectory: needs a CUDA device (there is no CPU fallback)")
    run(a.config, torch.float64 if a.dtype == "f64" else torch.float32, a.nsteps, not a.no_observables)  # warm-up
    print(json.dumps(run(a.config, torch.float64 if a.dtype == "f64" else torch.float32, a.nsteps,
                         not a.no_observables)), flush=True)


if __name__ == "__main__":
    main(sys.argv[1:])
