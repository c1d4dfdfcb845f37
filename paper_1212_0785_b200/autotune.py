"""Auto-tuning of launch parameters with a persisted table (section 4:
"QDP-JIT executes each kernel and measures the execution time as a function of N_t and determines the best
value and stores it in a database").

    python -m paper_1212_0785_b200.autotune --dims 32,32,32,64 --dtype f64 [--out tune.json] [--csv sweep.csv]

For the site-local kernels (link update, momentum update) the parameter is the paper's N_t, threads per
block; for the stencil kernel (gauge force) it is the kernel variant and the 4-D tile a block owns.  Every
candidate is timed through the public calls with CUDA events (median of `reps` after warm-up) on fields
larger than L2 where the lattice allows; the best goes into the library's database (qcd_tune_set), and the
whole table — winners and every measured candidate, the data behind the paper's Fig. 1 — can be written to
JSON and loaded again later (`load`).  Only launch parameters change; results stay within rounding order.
"""
import argparse
import itertools
import json
import sys

import torch

from . import binding as qcd

SITE_LOCAL_THREADS = (32, 64, 96, 128, 160, 192, 224, 256)
FORCE_BLOCK_SITES = 128  # threads per block of the stencil kernels (one thread per site of the subset)
FORCE_VARIANTS = ("plane", "staple")


def _divisors(n, even=False):
    return [d for d in range(1, n + 1) if n % d == 0 and (not even or d % 2 == 0)]


def force_tiles(dims, limit_sites, keep=12):
    """4-D tiles that divide the lattice and fill the block — the largest site count <= limit, and the next
    smaller one when it allows whole x rows (48-wide lattices: 96-site tiles of whole rows against 128-site tiles
    of 16-wide rows) — longest x rows first (coalescing), then the smallest surface"""
    cands = []
    for t in itertools.product(_divisors(dims[0], True), _divisors(dims[1]), _divisors(dims[2]), _divisors(dims[3])):
        sites = t[0] * t[1] * t[2] * t[3]
        if sites <= limit_sites:
            cands.append((sites, t))
    if not cands:
        return []
    top = max(s for s, _ in cands)
    full = [t for s, t in cands if s == top]
    full.sort(key=lambda t: (-min(t[0], 32), sum(1.0 / x for x in t)))
    rows = [t for s, t in cands if t[0] == dims[0] and s >= 0.75 * top and s != top]
    rows.sort(key=lambda t: (-t[0] * t[1] * t[2] * t[3], sum(1.0 / x for x in t)))
    return full[:keep] + rows[:4]


def _time(fn, warm=3, reps=10):
    for _ in range(warm):
        fn()
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(reps + 1)]
    for i in range(reps):
        ev[i].record()
        fn()
    ev[reps].record()
    torch.cuda.synchronize()
    ts = sorted(ev[i].elapsed_time(ev[i + 1]) for i in range(reps))
    return ts[reps // 2]


def tune(dims, dtype=torch.float64, subset=qcd.ALL, beta=6.0, eps=0.02, sigma=0.2, reps=10, verbose=True):
    """measure every candidate for the three tunable kernels on lattice `dims`; set the winners in the library;
    return the table (list of dict entries, one per kernel)"""
    prec = qcd.F64 if dtype == torch.float64 else qcd.F32
    lat = qcd.Lattice(dims)
    U, P, F = lat.new_matrix_field(dtype), lat.new_matrix_field(dtype), lat.new_matrix_field(dtype)
    qcd.qcd_hot_start(lat, U, 1234, sigma)
    qcd.qcd_mom_refresh(lat, P, 99)
    F.copy_(P)
    entries = []

    def record(kernel, name, cands):
        best = min(cands, key=lambda c: c["ms"])
        entries.append({"dims": list(dims), "prec": "f64" if prec == qcd.F64 else "f32", "subset": subset,
                        "kernel": name, "best": best, "candidates": cands})
        if verbose:
            for c in cands:
                print(f"{name:12s} {c['variant'] or '':8s} tile={c['tile']} threads={c['threads']:4d} "
                      f"{c['ms']:9.4f} ms{'  <- best' if c is best else ''}", flush=True)

    # stencil kernel: variant x tile
    cands = []
    for v in FORCE_VARIANTS:
        npar = 2 if subset == qcd.ALL else 1
        for tile in force_tiles(dims, FORCE_BLOCK_SITES * 2 // npar):
            try:
                qcd.qcd_tune_set(lat, prec, subset, qcd.KERNEL_FORCE, qcd.FORCE_VARIANTS.index(v), tile)
            except qcd.QcdError:
                continue
            ms = _time(lambda: qcd.qcd_force_mom_update(lat, U, P, beta, eps, subset=subset), reps=reps)
            cands.append({"variant": v, "tile": list(tile), "threads": 0, "ms": ms})
    record(qcd.KERNEL_FORCE, "force", cands)
    b = entries[-1]["best"]
    qcd.qcd_tune_set(lat, prec, subset, qcd.KERNEL_FORCE, qcd.FORCE_VARIANTS.index(b["variant"]), b["tile"])
    # site-local kernels: N_t
    qcd.qcd_mom_refresh(lat, P, 99)
    for kernel, name, fn in (
            (qcd.KERNEL_LINK_UPDATE, "link_update", lambda: qcd.qcd_link_update(lat, P, U, eps * 1e-3, reunit=True, subset=subset)),
            (qcd.KERNEL_MOM_UPDATE, "mom_update", lambda: qcd.qcd_mom_update(lat, F, P, 1e-6, subset=subset))):
        cands = []
        for nt in SITE_LOCAL_THREADS:
            qcd.qcd_tune_set(lat, prec, subset, kernel, threads=nt)
            cands.append({"variant": None, "tile": None, "threads": nt, "ms": _time(fn, reps=reps)})
        record(kernel, name, cands)
        qcd.qcd_tune_set(lat, prec, subset, kernel, threads=entries[-1]["best"]["threads"])
    return entries


def save(entries, path):
    dev = torch.cuda.get_device_name() if torch.cuda.is_available() else "unknown"
    with open(path, "w") as f:
        json.dump({"device": dev, "library": qcd.lib.qcd_version().decode(), "entries": entries}, f, indent=1)


def load(path):
    """apply the winners of a saved table to the library's database; returns the number of entries set"""
    kernels = {"force": qcd.KERNEL_FORCE, "link_update": qcd.KERNEL_LINK_UPDATE, "mom_update": qcd.KERNEL_MOM_UPDATE}
    n = 0
    for e in json.load(open(path))["entries"]:
        lat = qcd.Lattice(e["dims"])
        prec = qcd.F64 if e["prec"] == "f64" else qcd.F32
        b = e["best"]
        if e["kernel"] == "force":
            qcd.qcd_tune_set(lat, prec, e["subset"], kernels["force"], qcd.FORCE_VARIANTS.index(b["variant"]), b["tile"])
        else:
            qcd.qcd_tune_set(lat, prec, e["subset"], kernels[e["kernel"]], threads=b["threads"])
        n += 1
    return n


def write_csv(entries, path):
    with open(path, "w") as f:
        f.write("dims,prec,subset,kernel,variant,tile,threads,ms,best\n")
        for e in entries:
            for c in e["candidates"]:
                tile = "x".join(map(str, c["tile"])) if c["tile"] else ""
                f.write(f"{'x'.join(map(str, e['dims']))},{e['prec']},{e['subset']},{e['kernel']},{c['variant'] or ''},"
                        f"{tile},{c['threads']},{c['ms']:.5f},{int(c is e['best'])}\n")


def main(argv=None):
    ap = argparse.ArgumentParser(description=__doc__.split("\n\n")[0])
    ap.add_argument("--dims", default="32,32,32,64")
    ap.add_argument("--dtype", default="f64", choices=["f64", "f32"])
    ap.add_argument("--subset", type=int, default=qcd.ALL, choices=[qcd.ALL, qcd.EVEN, qcd.ODD])
    ap.add_argument("--reps", type=int, default=10)
    ap.add_argument("--out", help="write the table (JSON) here")
    ap.add_argument("--csv", help="write every measured candidate (CSV) here")
    a = ap.parse_args(argv)
    if not torch.cuda.is_available():
        raise SystemExit("autotune: needs a CUDA device")
    dims = tuple(int(x) for x in a.dims.split(","))
    entries = tune(dims, torch.float64 if a.dtype == "f64" else torch.float32, a.subset, reps=a.reps)
    if a.out:
        save(entries, a.out)
    if a.csv:
        write_csv(entries, a.csv)


if __name__ == "__main__":
    main(sys.argv[1:])
