"""Shared helpers of the GPU parity tests: run the CUDA path (through the C ABI binding) and the
CPU oracle on the same seeded inputs and compare element by element.

Tolerances (BASELINE.json north_star): fp64 1e-10 relative; fp32 mode 1e-5 on the energy and 1e-4
RMS on the forces. The fp32 outputs the north star does not bound are held to the bounds DESIGN.md
section 3 derives from the arithmetic (FP32_BOUNDS, each within 5x of the worst value measured on
the B200 over all fp32 cases). "Relative" is taken against the natural scale of each output
(DESIGN.md "Tolerances"): |U| for the energy, max|V| for potentials, reading F1's scale for forces
(max of the largest force and the largest single pair force, so that a perfect crystal with F = 0
is not divided by zero), max|Q| / max|E| for grids (not below one particle's charge, resp. its
potential at the cutoff), max(|W|, |U|) for the virial.
"""
from __future__ import annotations

import numpy as np

FP64_RTOL = 1e-10
FP32_ENERGY_RTOL = 1e-5
FP32_FORCE_RMS_RTOL = 1e-4
# fp32 mode, outputs without a north-star bound (DESIGN.md section 3 "Tolerances"): key -> bound;
# "Q" / "E" apply to the grids of every tiled level
FP32_BOUNDS = {"force_rms": 1e-5, "force_max": 2e-5, "potential_max": 2e-5, "virial": 2e-5, "Q": 6e-6, "E": 3e-4}


def run_oracle(w, mu=4, want_virial=True):
    from oracle import Oracle
    orc = Oracle(w.box, w.periodic, w.h, w.a, w.p, w.levels, mu=mu)
    res = orc.evaluate(w.positions, w.charges, want_virial=want_virial)
    res["oracle"] = orc
    return res


def run_gpu(w, precision=None, mu=-1, want_virial=True):
    from paper_2510_05961_b200 import msm
    return msm.evaluate_workload(w, precision=precision, mu=mu, want_virial=want_virial)


def force_scale(w, ref_forces):
    """Reading F1: max(max_i |F_i|_inf, largest single pair force max_ij |q_i q_j| / r_min^2
    bounded below by the pair force at the typical spacing)."""
    fmax = float(np.abs(ref_forces).max()) if ref_forces.size else 0.0
    n = len(w.charges)
    if n < 2:
        return max(fmax, 1.0)
    vol = 1.0
    for b in w.box:
        vol *= b
    dbar = (vol / n) ** (1.0 / 3.0)
    qmax = float(np.abs(w.charges).max())
    return max(fmax, qmax * qmax / (dbar * dbar))


def compare(w, gpu, ref, precision="fp64", check_grids=True):
    """Assert parity of one evaluation. Returns a dict of the measured relative errors."""
    out = {}
    U, Ur = gpu["energy"], ref["energy"]
    F, Fr = gpu["forces"], ref["forces"]
    V, Vr = gpu["potentials"], ref["potentials"]
    escale = max(abs(Ur), 1e-300)
    out["energy"] = abs(U - Ur) / escale
    fs = force_scale(w, Fr)
    out["force_max"] = float(np.abs(F - Fr).max()) / fs if F.size else 0.0
    frms = float(np.sqrt(np.mean(Fr ** 2))) if F.size else 0.0
    out["force_rms"] = float(np.sqrt(np.mean((F - Fr) ** 2))) / max(frms, fs * 1e-3) if F.size else 0.0
    vs = max(float(np.abs(Vr).max()), 1e-300) if V.size else 1.0
    out["potential_max"] = float(np.abs(V - Vr).max()) / vs if V.size else 0.0
    if gpu.get("virial") is not None and ref.get("virial") is not None:
        ws = max(float(np.abs(ref["virial"]).max()), abs(Ur), 1e-300)
        out["virial"] = float(np.abs(gpu["virial"] - ref["virial"]).max()) / ws
    if check_grids:
        plan, orc = gpu["plan"], ref["oracle"]
        for l in range(1, plan.info.n_tiled + 1):
            for kind in ("Q", "E"):
                g, r = plan.debug_grid(l, kind), orc.grid(l, kind)
                assert g.shape == r.shape, (l, kind, g.shape, r.shape)
                # floor of the scale: one particle's charge (Q) / its potential at the cutoff (E), so
                # that grids holding only round-off (coarse levels of a perfect crystal) compare
                qmax = float(np.abs(w.charges).max()) if len(w.charges) else 1.0
                floor = qmax if kind == "Q" else qmax / w.a
                s = max(float(np.abs(r).max()), floor)
                out[f"{kind}{l}"] = float(np.abs(g - r).max()) / s
    if precision == "fp64":
        for k, v in out.items():
            assert v <= FP64_RTOL, f"{w.name}: {k} relative error {v:.3e} > {FP64_RTOL:g} ({out})"
    else:
        assert out["energy"] <= FP32_ENERGY_RTOL, f"{w.name}: fp32 energy {out}"
        assert out["force_rms"] <= FP32_FORCE_RMS_RTOL, f"{w.name}: fp32 force rms {out}"
        for k, v in out.items():
            if k == "energy":
                continue
            bound = FP32_BOUNDS[k[0] if k[0] in "QE" and k[1:].isdigit() else k]
            assert v <= bound, f"{w.name}: fp32 {k} {v:.3e} > {bound:g} ({out})"
    return out


def small_workload(kind, n, seed, p=4, precision="fp64"):
    """Small seeded cases with the structure of the configs (several tiles + ragged tails)."""
    from paper_2510_05961_b200.workloads import Workload
    rng = np.random.default_rng(seed)
    if kind == "open":
        box = (17.3, 13.1, 21.7)
        pos = rng.random((n, 3)) * np.array(box)
        q = rng.uniform(-1, 1, n)
        w = Workload(f"small_open_{n}", pos, q, box, (0, 0, 0), h=1.9, a=5.0, p=p, levels=3)
    elif kind == "periodic":
        box = (23.0, 23.0, 23.0)
        pos = rng.random((n, 3)) * np.array(box)
        q = rng.uniform(-1, 1, n); q -= q.mean()
        w = Workload(f"small_periodic_{n}", pos, q, box, (1, 1, 1), h=1.5, a=6.0, p=p, levels=2)
    elif kind == "slab":
        box = (26.0, 26.0, 9.0)
        pos = rng.random((n, 3)) * np.array(box)
        q = rng.uniform(-1, 1, n); q -= q.mean()
        w = Workload(f"small_slab_{n}", pos, q, box, (1, 1, 0), h=1.6, a=6.5, p=p, levels=2)
    else:
        raise KeyError(kind)
    return w.as_precision(precision)
