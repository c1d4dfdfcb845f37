"""One molecular-dynamics trajectory of a BASELINE config on the GPU, with per-step observables.

    python -m paper_1212_0785_b200.trajectory --config 5 --dtype f64 [--nsteps 20] [--no-observables]

Momentum refresh and hot start from the counter-based generator, H before, a leapfrog
trajectory (PAPER.md:17 operations; integrator R6), H after, dH.  With observables (default) every step's
momentum update is `qcd_force_mom_update_sums`, so the plaquette and the kinetic energy of every step come
out of the force kernel itself (no extra pass over the fields); without, the plain fused kernels run.
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
    V = lat.V
    U, P = lat.new_matrix_field(dtype), lat.new_matrix_field(dtype)
    ws = lat.new_workspace()
    qcd.qcd_hot_start(lat, U, seed, c["sigma"])
    qcd.qcd_mom_refresh(lat, P, seed)
    obs = torch.zeros((n + 2, 2), dtype=torch.float64, device="cuda")  # rows: start, after each step's kick

    def energy(row):
        qcd.qcd_plaquette(lat, U, obs[row, 0:1], None, ws)
        qcd.qcd_sum(lat, qcd.SUM_NORM2, 72, P, obs[row, 1:2], ws)

    energy(0)
    stream = torch.cuda.current_stream()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record(stream)
    # O11: P += eps/2 F; n x { U <- reunit(exp(i eps P) U); P += eps F (eps/2 on the last) }
    qcd.qcd_force_mom_update(lat, U, P, beta, 0.5 * eps)
    for k in range(n):
        qcd.qcd_link_update(lat, P, U, eps, reunit=True)
        step_eps = 0.5 * eps if k == n - 1 else eps
        if observables:
            qcd.qcd_force_mom_update_sums(lat, U, P, beta, step_eps, obs[k + 1], ws)
        else:
            qcd.qcd_force_mom_update(lat, U, P, beta, step_eps)
    e1.record(stream)
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1)
    energy(n + 1)  # stand-alone reductions at the end: must agree with the by-products of the last kick
    o = obs.cpu().numpy()

    def H(row):
        return float(o[row, 1] + beta * 6 * V * (1 - o[row, 0]))

    rb = 8 if dtype == torch.float64 else 4
    peak = 6532.5
    pk = os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "MEASURED_PEAKS.json")
    if os.path.exists(pk):
        peak = float(json.load(open(pk))["hbm_gbs"])
    gbs = 432 * rb * V * n / (ms * 1e-3) / 1e9
    line = {"config": config, "dims": list(dims), "dtype": "f64" if rb == 8 else "f32", "nsteps": n, "eps": eps,
            "beta": beta, "observables_every_step": observables, "ms": ms, "ms_per_step": ms / n,
            "site_updates_per_s": V * n / (ms * 1e-3), "step_hbm_gbs": gbs, "step_frac_of_hbm_peak": gbs / peak,
            "plaq_start": float(o[0, 0]), "K_start": float(o[0, 1]), "H_start": H(0),
            "plaq_end": float(o[n + 1, 0]), "K_end": float(o[n + 1, 1]), "H_end": H(n + 1), "dH": H(n + 1) - H(0),
            "K_per_16V_start": float(o[0, 1] / (16 * V))}
    if observables:
        line["dH_from_fused_sums"] = H(n) - H(0)
        line["per_step_plaq_K"] = [[float(a), float(b)] for a, b in o[1:n + 1]]
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
