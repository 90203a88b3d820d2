#!/usr/bin/env python
"""bench.py -- times the whole hot path of the Lanczos full-frequency GW method on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config i] [--full] [--impl ours|reference]

One "step" = one pass of the whole path over one synthetic problem of
BASELINE.json:configs[i] (default configs[4], the largest single-GPU configuration): start vectors, Lanczos
steps of the chains in blocks (each step one Casida block product plus the recurrence), Ritz/continued-fraction
evaluation of Sigma^c on the omega grid and the sum over chains.  For configs 2-4 a pass is BOUNDED so that the
default run ends within minutes: one block of B chains x L_bench Lanczos steps (PASS below; named in
config.workload / chains / lanczos_steps); chain-steps/s does not depend on L in steady state (every step is the same
block product) and the S1/S6 overhead of the short pass is inside the timed region.  --full runs all chains x full L.
  value   = Lanczos chain-steps/s, whole job, inputs resident in HBM (device-pointer C-ABI calls)
  e2e     = the same through the host-pointer C-ABI calls: every step uploads orbitals, energies, the
            Coulomb kernel and the chain list from pinned host memory and reads alpha/beta/Sigma back
  roofline= the dominant kernel (a Khatri-Rao GEMM) against the FP64 tensor (DMMA) peak
  cpu_baseline = the NumPy oracle (oracle/gw_oracle.py), as it stands, on the host cores
N > 1: independent replicas, one per GPU ("replicas only"); value sums their chain-steps over the max time.
Prints ONE JSON line on rank 0.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

METRIC = "lanczos_chain_steps_per_s"
UNIT = "chain-steps/s"
L2_FLUSH_BYTES = 512 << 20
# bounded pass per config: (chains, Lanczos steps); None = the whole config (all chains x full L)
PASS = {0: None, 1: None, 2: (256, 60), 3: (256, 20), 4: (128, 10)}


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=None,
                    help="index into BASELINE.json:configs (default 4, the largest; 2 with --sharded-state)")
    ap.add_argument("--full", action="store_true", help="all chains x full L of the config instead of the bounded pass")
    ap.add_argument("--chains", type=int, default=0, help="override the number of chains of a pass (marks the line)")
    ap.add_argument("--tdc", default="", metavar="NK,NV,NC,NMU",
                    help="context run, not the bench line: the complex-orbital Tamm-Dancoff variant (SURVEY 8(f)-3) on a "
                         "synthetic periodic problem of that shape, e.g. 4,64,1024,6144; block = --chains (default 128), "
                         "L = --lanczos-steps (default 10)")
    ap.add_argument("--block", type=int, default=0, help="with --paper-setting: chains per block (default 256)")
    ap.add_argument("--rpa", action="store_true",
                    help="with --tdc: the full RPA for complex orbitals (pseudo-Hermitian Lanczos on C^RPA(q), PAPER.md:159): every "
                         "chain is a pair [x; y] = two GEMM columns, one product with Omega^ per step")
    ap.add_argument("--sym", type=int, default=-1, metavar="NGEN",
                    help="context run, not the bench line: the point-group symmetry blocks of C (SURVEY 8(f)-4, PAPER.md:128) for an "
                         "abelian group of order 2^NGEN on a synthetic system with the sizes of --config (default 4): one block "
                         "of chains x L Lanczos steps inside the pair-irrep block gamma = 1")
    ap.add_argument("--sharded-state", action="store_true",
                    help="SURVEY 8(f)-2 arm, its own line: the N_v+N_c chains of ONE state partitioned over the ranks "
                         "(runtime.shard_range), one NCCL all-reduce of the omega grid; strong scaling")
    ap.add_argument("--isdf", default="", metavar="NGRID,NORB,NMU[,SEED]",  # SEED < 0: pick the first well-conditioned stride-point set
                    help="context run, not the bench line: the ISDF front end (SURVEY 8(f)-4; gwl_isdf_build) on NORB particle-in-"
                         "a-box orbitals on an NGRID^3 grid with NMU interpolation points, e.g. 40,256,1024: "
                         "seconds per build, flop model and fraction of the DMMA peak")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--lanczos-steps", type=int, default=0, help="override L (for profiling runs only; marks the line)")
    ap.add_argument("--reorth", action="store_true",
                    help="two-pass full reorthogonalisation on (not the bench workload; marks the line)")
    ap.add_argument("--paper-setting", default="", metavar="NV,NC,NMU",
                    help="context run, not the bench line: one whole quasiparticle state (all N_v+N_c chains, Sigma^x, "
                         "E(omega)=omega) with the paper's parameters N_iter = 8, g = 7 (PAPER.md:145) on a synthetic "
                         "problem of that shape, e.g. 210,1520,7000 for Si86H76 (Table I)")
    return ap.parse_args()


def pass_shape(args, cfg):
    """(chains, L) of one timed pass."""
    i = cfg_index(cfg)
    nch, L = (cfg.n_chains, cfg.steps) if (args.full or PASS[i] is None) else PASS[i]
    if args.lanczos_steps:
        L = args.lanczos_steps
    if args.chains:
        nch = min(args.chains, cfg.n_chains)
    return nch, L


def workload_config(cfg, n_gpus, L, nch=None):
    nch = cfg.n_chains if nch is None else nch
    i = cfg_index(cfg)
    what = f"BASELINE.json:configs[{i}] {cfg.name}"
    if (nch, L) != (cfg.n_chains, cfg.steps):
        what += (f"; bounded pass: {nch} chains (blocks of {cfg.block}) x {L} Lanczos steps of the config's "
                 f"{cfg.n_chains} x {cfg.steps}, S1 + S2-S4 + S5-S7 on the full omega grid")
    return {"workload": what, "n_v": cfg.n_v, "n_c": cfg.n_c,
            "n_mu": cfg.n_mu, "n_vc": cfg.n_vc, "chains": nch, "block": cfg.block, "lanczos_steps": L,
            "n_omega": cfg.n_omega, "eta_eV": cfg.eta, "mode": "direct (Op = C), reorth off",
            "parallelism": "single GPU" if n_gpus == 1 else f"{n_gpus} independent replicas",
            "l2": f"flushed between timed steps ({L2_FLUSH_BYTES >> 20} MiB write)", "seed": 0}


def cfg_index(cfg):
    from paper_2310_20103_b200 import synth
    return synth.CONFIGS.index(cfg)


# ------------------------------------------------------------------------------------------------
def oracle_sample(prob, n_chains, L):
    """Runs the oracle, as it stands, on `n_chains` chains x `L` steps of the workload; returns seconds."""
    from oracle import gw_oracle as orc
    t0 = time.perf_counter()
    orc.run_chains(prob.phi_v, prob.phi_c, prob.eps_v, prob.eps_c, prob.V, prob.n_idx[:n_chains],
                   prob.m_idx[:n_chains], L, prob.omega, prob.cfg.eta, reorth=False)
    return time.perf_counter() - t0


def host_threads():
    try:
        from threadpoolctl import threadpool_info
        n = [d.get("num_threads", 1) for d in threadpool_info() if d.get("user_api") == "blas"]
        if n:
            return int(max(n))
    except Exception:
        pass
    return os.cpu_count() or 1


def cpu_baseline(prob, nch_pass, L_pass, budget_s=12.0):
    """Oracle timed on a bounded sample of the same workload (about 10-30 s of host work)."""
    t1 = oracle_sample(prob, 1, 2)                 # calibration (also warms BLAS)
    per = max(t1 / 2.0, 1e-6)
    total = max(4, min(int(budget_s / per), nch_pass * L_pass))
    L = max(2, min(L_pass, 20, total))
    nch = max(1, min(nch_pass, total // L))
    t = oracle_sample(prob, nch, L)
    return {"value": nch * L / t, "unit": UNIT, "cores": host_threads(), "kind": "oracle",
            "sample": f"{nch} chains x {L} Lanczos steps of the same workload + Sigma on the full omega grid, "
                      f"NumPy/SciPy FP64, {t:.1f} s", "host_cpus": os.cpu_count()}


def run_reference(args):
    """--impl reference: the oracle alone, on the host cores (this tier has no reference code to install)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from paper_2310_20103_b200 import synth
    cfg = synth.CONFIGS[args.config]
    nch_pass, L_pass = pass_shape(args, cfg)
    prob = synth.make_problem(cfg)
    _ = prob.V
    t1 = oracle_sample(prob, 1, 2)
    per = max(t1 / 2.0, 1e-6)
    budget = 150.0 / max(args.steps + args.warmup, 1)        # whole run within a few minutes
    total = max(2, int(budget / per))
    L = max(2, min(L_pass, 20, total))
    nch = max(1, min(nch_pass, total // L))
    for _ in range(args.warmup):
        oracle_sample(prob, nch, L)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle_sample(prob, nch, L)
    el = time.perf_counter() - t0
    val = args.steps * nch * L / el
    sample = f"each step = {nch} chains x {L} Lanczos steps + Sigma on the omega grid (bounded sample of the workload)"
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * el / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": workload_config(cfg, args.gpus, L_pass, nch_pass),
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": host_threads(), "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def run_paper_setting(args):
    """One quasiparticle state the way the paper runs it: Lanczos on p_g(C), g = 7,
    N_iter = 8, one chain per n = 1..N_v+N_c, then Sigma^x and the Newton-Raphson solve.  Context for BASELINE.md's
    Table I quotes (the paper's wall times include the CPU-only ISDF step and real data; this is the hot path only, on
    synthetic inputs of the same shape).  The fitting range comes from a 24-step Lanczos estimate of the top of the
    spectrum (polyfit.range_from_spectrum), inside the timed state."""
    import numpy as np
    import torch

    from paper_2310_20103_b200 import gwl, polyfit, synth

    n_v, n_c, n_mu = (int(x) for x in args.paper_setting.split(","))
    g, n_iter, block = 7, 8, (args.block or 256)
    torch.cuda.set_device(0)
    dev = torch.device("cuda", 0)
    gwl.load_library()
    n_orb = n_v + n_c
    m = n_v - 1                                                   # the HOMO
    gord = 1 << max(args.sym, 0)
    if args.sym >= 0:
        # the same shape with an abelian point group of order 2^NGEN (the paper's clusters are symmetric and its
        # Table I times use that): orbitals spread evenly over the irreps, N_mu / g wedge points
        split = lambda n: [n // gord + (1 if a < n % gord else 0) for a in range(gord)]
        prob = synth.make_symmetric(args.sym, split(n_v), split(n_c), n_mu // gord, box=25.0, seed=0, n_omega=401)
        ctx = gwl.SymContext(args.sym, prob.nv_irrep, prob.nc_irrep, prob.n_w)
        phi_v, phi_c, kern = prob.phi_v_w, prob.phi_c_w, prob.V_wf
    else:
        prob = synth.make_custom(n_v, n_c, n_mu, box=25.0, seed=0, n_omega=401)
        ctx = gwl.Context(n_v, n_c, n_mu)
        phi_v, phi_c, kern = prob.phi_v, prob.phi_c, prob.V
    stream = torch.cuda.current_stream()
    ctx.set_stream(stream.cuda_stream)
    ctx.set_orbitals(phi_v, phi_c)
    ctx.set_energies(prob.eps_v, prob.eps_c)
    ctx.set_kernel(kern)
    ctx.set_pointer_mode(1)
    ctx.set_profiling(0)
    om = torch.from_numpy(prob.omega).to(dev)
    sc = torch.empty(1, len(prob.omega), 2, dtype=torch.float64, device=dev)
    sx = torch.empty(1, dtype=torch.float64, device=dev)
    out = (torch.empty(1, dtype=torch.float64, device=dev), torch.empty(1, dtype=torch.float64, device=dev),
           torch.empty(1, dtype=torch.int32, device=dev))
    rng = [0.0, 0.0]
    n_probe = [0]

    def state():
        ctx.set_polynomial(0)
        if args.sym >= 0:   # one fitting range for all blocks: the largest upper bound over the blocks
            d_min = float(prob.eps_c.min() - prob.eps_v.max())
            hi, n_probe[0] = 0.0, 0
            for gamma in range(gord):
                try:
                    ctx.select(gamma)
                except gwl.GwlError:
                    continue                                       # a block without pairs
                hi = max(hi, ctx.spectrum_bounds(24)[1])
                n_probe[0] += 1
            lo, hi = 0.8 * d_min * d_min, 1.02 * hi
        else:
            lo, hi = polyfit.range_from_spectrum(ctx, prob.eps_v, prob.eps_c, steps=24)
            n_probe[0] = 1
        rng[:] = [lo, hi]
        ctx.set_polynomial(g, polyfit.sqrt_chebyshev(g, lo, hi), lo, hi)
        ctx.selfenergy_state(m, n_iter, block, 0, om, 0.68, out=sc[0])        # delta = 0.05 Ry
        ctx.exchange([m], out=sx)
        ctx.qp_solve([prob.eps_v[m]], [-9.0], sx, sc, om, out=out)

    for _ in range(args.warmup):          # --warmup 0 is accepted here: a big shape takes tens of minutes per pass
        state()
    torch.cuda.synchronize()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    n0 = ctx.get_launch_count()
    for a, b in ev:
        a.record(stream)
        state()
        b.record(stream)
    torch.cuda.synchronize()
    sec = sum(a.elapsed_time(b) for a, b in ev) * 1e-3 / args.steps
    launches = int((ctx.get_launch_count() - n0) / args.steps)
    # one more state with an event pair around every launch: where the time goes (not part of the timed value)
    ctx.set_profiling(2)
    state()
    kt = ctx.get_kernel_times()
    ctx.set_profiling(0)
    tot = sum(v[0] for v in kt.values())
    share = {k: round(v[0] / tot, 4) for k, v in kt.items() if v[1]}
    per_launch_ms = {k: round(v[0] / v[1], 4) for k, v in kt.items() if v[1]}
    if args.sym >= 0:   # reduced operator: chains of irrep a run in block a ^ irrep(m) on n_w points
        irr = np.concatenate([prob.irrep_v, prob.irrep_c])
        pairs = [int(((prob.irrep_v[:, None] ^ prob.irrep_c[None, :]) == gam).sum()) for gam in range(gord)]
        per_vec = [4.0 * prob.n_w * pairs[gam] + 2.0 * prob.n_w * prob.n_w for gam in range(gord)]
        flop = sum(per_vec[int(irr[n] ^ irr[m])] for n in range(n_orb)) * n_iter * g + 24 * sum(per_vec)
    else:
        flop = (n_orb * n_iter * g + 24) * (4.0 * n_mu * n_v * n_c + 2.0 * n_mu * n_mu)
    line = {"metric": "seconds_per_quasiparticle_state", "value": sec, "unit": "s", "higher_is_better": False,
            "n_gpus": 1, "steps": args.steps, "warmup": args.warmup, "dtype": "f64", "data": "synthetic",
            "config": {"workload": "paper setting: N_iter = 8, g = 7 (PAPER.md:145), all N_v+N_c chains of one state, "
                                   "Sigma^x, Newton-Raphson; fitting range from a 24-step Lanczos bound (PAPER.md:284)",
                       "n_v": n_v, "n_c": n_c, "n_mu": n_mu, "chains": n_orb, "block": block,
                       "fit_range_eV2": rng, "point_group_order": gord,
                       "symmetry": ("blocks of C by pair irrep (gwl_sym_*, PAPER.md:128), wedge of %d points" % (n_mu // gord))
                       if args.sym >= 0 else "none"},
            "c_applies": n_orb * n_iter * g + 24 * n_probe[0], "tflops_flop_model": flop / sec / 1e12,
            "gpu_launches": launches, "kernel_time_share": share, "kernel_ms_per_launch": per_launch_ms,
            "e_qp_eV": float(out[0].item()), "z": float(out[1].item()),
            "note": "context only: hot path on synthetic inputs; the paper's Table I wall times include ISDF on CPUs"}
    print(json.dumps(line), flush=True)
    ctx.close()


def run_tdc(args):
    """Complex-orbital Tamm-Dancoff variant (gwl_tdc_*): one block of chains x L Lanczos steps on the Hermitian A(q) + Sigma,
    with the complex Khatri-Rao GEMMs against the DMMA roofline (8 N_mu N_kvc B real flop per launch: 4 real multiply-adds
    per complex one)."""
    import torch

    from paper_2310_20103_b200 import gwl, synth

    n_k, n_v, n_c, n_mu = (int(x) for x in args.tdc.split(","))
    nch = args.chains or 128
    L = args.lanczos_steps or 10
    torch.cuda.set_device(0)
    dev = torch.device("cuda", 0)
    gwl.load_library()
    p = synth.make_periodic(n_k, n_v, n_c, n_mu, box=20.0, seed=0, n_omega=401, n_chains=nch)
    ctx = gwl.TdcContext(n_k, n_v, n_c, n_mu, 1)
    stream = torch.cuda.current_stream()
    ctx.set_stream(stream.cuda_stream)
    ctx.set_orbitals(p.psi_v, p.psi_cq)
    ctx.set_energies(p.eps_v, p.eps_cq)
    ctx.set_kernel(p.V)
    if args.rpa:
        ctx.set_approximation(gwl.GWL_RPA)
    ctx.set_chains(p.chains)
    ctx.set_pointer_mode(1)
    ctx.set_profiling(0)
    om = torch.from_numpy(p.omega).to(dev)
    ssum = torch.empty(len(p.omega), 2, dtype=torch.float64, device=dev)
    peak = gwl.probe_fp64_peak(0)
    cols = 2 * nch if args.rpa else nch      # GEMM columns per block: a pair [x; y] is two columns

    def step():
        ctx.lanczos(nch, L, nch, 0, out=None)
        ctx.selfenergy(om, 0.1, out=(None, ssum))

    for _ in range(args.warmup):
        step()
    torch.cuda.synchronize()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    for a, b in ev:
        a.record(stream)
        step()
        b.record(stream)
    torch.cuda.synchronize()
    sec = sum(a.elapsed_time(b) for a, b in ev) * 1e-3 / args.steps
    ctx.set_profiling(2)
    step()
    kt = ctx.get_kernel_times()
    ctx.set_profiling(0)
    n_kvc = n_k * n_v * n_c
    fl = 8.0 * n_mu * n_kvc * cols
    per = {k: v[0] / v[1] for k, v in kt.items() if v[1]}
    line = {"metric": METRIC, "value": nch * L / sec, "unit": UNIT, "n_gpus": 1, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": 1e3 * sec, "higher_is_better": True, "dtype": "complex f64 (planar)", "data": "synthetic",
            "arm": ("complex RPA" if args.rpa else "tdc") + " (SURVEY 8(f)-3): context run, not the headline bench line",
            "config": {"workload": ("periodic RPA: pseudo-Hermitian Lanczos on C^RPA(q) in the Omega^ inner product, one block of "
                                    "chain pairs (2 GEMM columns per chain)" if args.rpa else
                                    "periodic Tamm-Dancoff: Lanczos on the Hermitian A(q), one block of chains"), "n_k": n_k,
                       "n_v": n_v, "n_c": n_c, "n_mu": n_mu, "n_kvc": n_kvc, "chains": nch, "lanczos_steps": L},
            "roofline": {"bound": "tensor", "peak": peak, "unit": "TFLOP/s",
                         "Kx": {"achieved": fl / (per["gemm_fwd_KX"] * 1e-3) / 1e12, "ms_per_launch": per["gemm_fwd_KX"]},
                         "KhW": {"achieved": fl / (per["gemm_bwd_KtW"] * 1e-3) / 1e12, "ms_per_launch": per["gemm_bwd_KtW"]},
                         "flop_per_launch": fl, "flop_model": "8 N_mu N_kvc B real flop (4 real multiply-adds per complex one), B = GEMM columns"},
            "kernel_time_share": {k: round(v[0] / sum(x[0] for x in kt.values()), 4) for k, v in kt.items() if v[1]}}
    line["roofline"]["Kx"]["frac"] = line["roofline"]["Kx"]["achieved"] / peak
    line["roofline"]["KhW"]["frac"] = line["roofline"]["KhW"]["achieved"] / peak
    print(json.dumps(line), flush=True)
    ctx.close()


def run_sym(args):
    """Symmetry blocks (gwl_sym_*): one block of chains x L steps inside one pair-irrep block of a system with the sizes of a
    BASELINE config and an abelian point group of order g; flop model of the REDUCED operator, (4 n_w N_pairs + 2 n_w^2) B per
    block product, next to what the same chains cost without the symmetry."""
    import numpy as np
    import torch

    from paper_2310_20103_b200 import gwl, synth

    cfg = synth.CONFIGS[2 if args.config is None else args.config]
    g = 1 << args.sym
    if cfg.n_v % g or cfg.n_c % g or cfg.n_mu % g:
        raise SystemExit("--sym: the config's N_v, N_c, N_mu must be divisible by the group order")
    nch = args.chains or min(cfg.block, cfg.n_v // g + cfg.n_c // g)
    L = args.lanczos_steps or 10
    torch.cuda.set_device(0)
    dev = torch.device("cuda", 0)
    gwl.load_library()
    p = synth.make_symmetric(args.sym, [cfg.n_v // g] * g, [cfg.n_c // g] * g, cfg.n_mu // g, box=cfg.box, seed=0,
                             n_omega=cfg.n_omega)
    gamma = 1 if g > 1 else 0
    irr = np.concatenate([p.irrep_v, p.irrep_c])
    m = 0
    n_idx = np.array([n for n in range(irr.size) if irr[n] ^ irr[m] == gamma][:nch], dtype=np.int32)
    nch = n_idx.size
    ctx = gwl.SymContext(args.sym, p.nv_irrep, p.nc_irrep, p.n_w)
    stream = torch.cuda.current_stream()
    ctx.set_stream(stream.cuda_stream)
    ctx.set_orbitals(p.phi_v_w, p.phi_c_w)
    ctx.set_energies(p.eps_v, p.eps_c)
    ctx.set_kernel(p.V_wf)
    n_pairs = ctx.select(gamma)
    ctx.set_chains(n_idx, np.full(nch, m, dtype=np.int32))
    ctx.set_pointer_mode(1)
    ctx.set_profiling(0)
    om = torch.from_numpy(p.omega).to(dev)
    ssum = torch.empty(len(p.omega), 2, dtype=torch.float64, device=dev)
    peak = gwl.probe_fp64_peak(0)

    def step():
        ctx.lanczos(nch, L, nch, 0, out=None)
        ctx.selfenergy(om, cfg.eta, out=(None, ssum))

    for _ in range(args.warmup):
        step()
    torch.cuda.synchronize()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    for a, b in ev:
        a.record(stream)
        step()
        b.record(stream)
    torch.cuda.synchronize()
    sec = sum(a.elapsed_time(b) for a, b in ev) * 1e-3 / args.steps
    ctx.set_profiling(2)
    step()
    kt = ctx.get_kernel_times()
    ctx.set_profiling(0)
    fl_block = (4.0 * p.n_w * n_pairs + 2.0 * p.n_w * p.n_w) * nch
    ms_mv = sum(kt[k][0] for k in ("gemm_fwd_KX", "gemm_V", "gemm_bwd_KtW", "splitk_reduce")) / (L + 0.5)
    line = {"metric": METRIC, "value": nch * L / sec, "unit": UNIT, "n_gpus": 1, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": 1e3 * sec, "higher_is_better": True, "dtype": "f64", "data": "synthetic",
            "arm": "sym (SURVEY 8(f)-4, PAPER.md:128): context run, not the headline bench line",
            "config": {"workload": f"symmetry block gamma = {gamma} of a system with the sizes of {cfg.name} and an abelian point "
                                   f"group of order {g}: one block of chains x L steps inside the block",
                       "group_order": g, "n_v": cfg.n_v, "n_c": cfg.n_c, "n_mu_full": cfg.n_mu, "n_mu_wedge": p.n_w,
                       "n_pairs_block": int(n_pairs), "n_vc_full": cfg.n_vc, "chains": int(nch), "lanczos_steps": L},
            "matvec": {"tflops": fl_block / (ms_mv * 1e-3) / 1e12, "frac_of_dmma_peak": fl_block / (ms_mv * 1e-3) / 1e12 / peak,
                       "ms_per_block_matvec": ms_mv, "flop_model": "(4 n_w N_pairs + 2 n_w^2) B (reduced operator)",
                       "flop_without_symmetry": cfg.flop_per_vector() * nch,
                       "flop_ratio": cfg.flop_per_vector() * nch / fl_block},
            "roofline": {"bound": "tensor", "peak": peak, "unit": "TFLOP/s"},
            "kernel_time_share": {k: round(v[0] / sum(x[0] for x in kt.values()), 4) for k, v in kt.items() if v[1]}}
    print(json.dumps(line), flush=True)
    ctx.close()


def cublas_dgemm_tflops(dev, n=8192, reps=3):
    """torch.matmul FP64 n^3 (cuBLAS DGEMM), best of `reps`: printed beside the DMMA probe as context."""
    import torch
    a = torch.randn(n, n, dtype=torch.float64, device=dev)
    b = torch.randn(n, n, dtype=torch.float64, device=dev)
    c = torch.matmul(a, b)
    torch.cuda.synchronize()
    best = None
    for _ in range(reps):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        torch.matmul(a, b, out=c)
        e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1)
        best = ms if best is None else min(best, ms)
    del a, b, c
    torch.cuda.empty_cache()
    return 2.0 * n ** 3 / (best * 1e-3) / 1e12


def run_isdf(args):
    """gwl_isdf_build timed end to end through the C ABI with HOST buffers (the call is synchronous:
    H2D of the orbitals and points, Z C^T and C C^T on the DMMA GEMM, Cholesky + solves, the dense Coulomb quadrature
    matrix G, G zeta and zeta^T G zeta on the DMMA GEMM, D2H of (alpha|beta)).  Prints its own JSON line."""
    import time

    import numpy as np
    import torch

    from paper_2310_20103_b200 import gwl, synth

    parts = [int(x) for x in args.isdf.split(",")]
    n_grid, n_orb, n_mu = parts[:3]
    seed = parts[3] if len(parts) > 3 else 1
    n_v = max(1, n_orb // 4)
    n_c = n_orb - n_v
    torch.cuda.set_device(0)
    gwl.load_library()
    r, phi, w = synth.box_orbitals(n_grid, n_orb)
    n_r = r.shape[0]
    if seed < 0:                                     # first stride-point set on which C C^T is safely positive definite
        for seed in range(16):
            idx = synth.stride_points(n_r, n_mu, seed)
            P = phi[idx] @ phi[idx].T
            ev = np.linalg.eigvalsh(P * P)
            if ev[0] > 0 and ev[-1] / ev[0] < 1e9:
                break
    idx = synth.stride_points(n_r, n_mu, seed)
    pv, pc = np.ascontiguousarray(phi[:, :n_v]), np.ascontiguousarray(phi[:, n_v:])
    peak = gwl.probe_fp64_peak(0)
    flop = {"ZCt": 2.0 * n_r * n_mu * n_orb, "cholesky": n_mu ** 3 / 3.0, "solves": 2.0 * n_mu ** 2 * n_r,
            "G_zeta": 2.0 * float(n_r) ** 2 * n_mu, "zetaT_G_zeta": 2.0 * n_r * float(n_mu) ** 2}
    times = []
    with gwl.Context(n_v, n_c, n_mu) as ctx:
        for i in range(args.warmup + args.steps):
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            _, V = ctx.isdf_build(pv, pc, r, w, 0.5, idx, want_zeta=False)
            torch.cuda.synchronize()
            if i >= args.warmup:
                times.append(time.perf_counter() - t0)
        launches = ctx.get_launch_count()
    t = float(np.median(times))
    total = sum(flop.values())
    line = {"arm": "isdf (SURVEY 8(f)-4): not the headline bench line", "metric": "isdf_build_seconds", "value": t, "unit": "s",
            "higher_is_better": False, "steps": args.steps, "warmup": args.warmup, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"gwl_isdf_build: {n_orb} box orbitals ({n_v} + {n_c}) on a {n_grid}^3 grid, n_r = {n_r}, "
                                   f"N_mu = {n_mu} stride points (seed {seed}), softened Coulomb quadrature (soft 0.5)",
                       "n_r": n_r, "n_orb": n_orb, "n_mu": n_mu},
            "flop_model": flop, "flop_total": total, "tflops_whole_call": total / t * 1e-12,
            "frac_of_dmma_peak_whole_call": total / t * 1e-12 / peak, "dmma_peak_tflops": peak,
            "host_bytes_in": int(pv.nbytes + pc.nbytes + r.nbytes + idx.nbytes), "host_bytes_out": int(V.nbytes),
            "gpu_launches_per_build": int(launches // (args.warmup + args.steps)),
            "V_checksum": float(np.abs(V).sum()), "V_asymmetry": float(np.abs(V - V.T).max() / np.abs(V).max())}
    print(json.dumps(line), flush=True)


SHARD_QUANTUM = 128   # chain shards are cut at multiples of the GEMM column tile (runtime.shard_range)


def run_sharded_state(args):
    """Sigma^corr_mm(omega) of ONE state with its N_v+N_c chains partitioned over the ranks
    (runtime.shard_range), direct mode, L steps each, ONE all-reduce (NCCL) of the omega grid.  Strong scaling:
    the total work is fixed as N grows.  Prints its own JSON line (not the headline bench line)."""
    import torch
    import torch.distributed as dist

    from paper_2310_20103_b200 import gwl, runtime, synth

    rank, local_rank, world = runtime.dist_env()
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    gwl.load_library()
    cfg = synth.CONFIGS[args.config]
    L = args.lanczos_steps or 8
    prob = synth.make_problem(cfg)
    n_orb = cfg.n_v + cfg.n_c
    m = cfg.n_v - 1
    stream = torch.cuda.current_stream()
    ctx = gwl.Context(cfg.n_v, cfg.n_c, cfg.n_mu)
    ctx.set_stream(stream.cuda_stream)
    ctx.set_orbitals(prob.phi_v, prob.phi_c)
    ctx.set_energies(prob.eps_v, prob.eps_c)
    ctx.set_kernel(prob.V)
    ctx.set_pointer_mode(1)
    ctx.set_profiling(0)
    om = torch.from_numpy(prob.omega).to(dev)
    local = runtime.gwl_local_sigma_sum(ctx, m, L, cfg.block, 0, om, cfg.eta)
    flush = torch.empty(L2_FLUSH_BYTES, dtype=torch.uint8, device=dev)
    for _ in range(args.warmup):
        runtime.sharded_sigma_state(local, n_orb, SHARD_QUANTUM)
    torch.cuda.synchronize()
    sampler = runtime.ClockSampler(local_rank).start()
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    pairs = []
    n0 = ctx.get_launch_count()
    for _ in range(args.steps):
        flush.zero_()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        sig = runtime.sharded_sigma_state(local, n_orb, SHARD_QUANTUM)
        e1.record(stream)
        pairs.append((e0, e1))
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    clocks = sampler.stop()
    elapsed = sum(a.elapsed_time(b) for a, b in pairs) * 1e-3
    lo, hi = runtime.shard_range(n_orb, rank, world, SHARD_QUANTUM)
    units, tmax = runtime.aggregate_throughput(float(args.steps) * (hi - lo) * L, elapsed, dev)
    if rank == 0:
        line = {"metric": METRIC, "value": units / tmax, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": 1e3 * tmax / args.steps, "higher_is_better": True,
                "scaling": "strong", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
                "arm": "sharded-state (SURVEY 8(f)-2): not the headline bench line",
                "config": {"workload": f"BASELINE.json:configs[{args.config}] {cfg.name}: Sigma^corr_mm of one state (HOMO), "
                                       f"all {n_orb} chains x {L} Lanczos steps, chains partitioned over {world} rank(s), "
                                       "one all-reduce of the omega grid", "n_v": cfg.n_v, "n_c": cfg.n_c,
                           "n_mu": cfg.n_mu, "chains": n_orb, "block": cfg.block, "lanczos_steps": L,
                           "n_omega": cfg.n_omega, "parallelism": f"chain-sharded x{world}",
                           "l2": f"flushed between timed steps ({L2_FLUSH_BYTES >> 20} MiB write)"},
                "clocks": clocks, "gpu_launches": int(ctx.get_launch_count() - n0),
                "allreduce_bytes_per_step": int(cfg.n_omega * 16) if world > 1 else 0,
                "chains_per_rank": [b - a for a, b in (runtime.shard_range(n_orb, r, world, SHARD_QUANTUM) for r in range(world))],
                "shard_quantum": SHARD_QUANTUM, "tile_efficiency": runtime.tile_efficiency(n_orb, world, SHARD_QUANTUM),
                "sigma_checksum": float(sig.abs().sum().item())}
        print(json.dumps(line), flush=True)
    ctx.close()
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


# ------------------------------------------------------------------------------------------------
def main():
    args = parse()
    if args.config is None:
        args.config = 2 if args.sharded_state else 4
    if args.impl == "reference":
        run_reference(args)
        return
    if args.paper_setting:
        run_paper_setting(args)
        return
    if args.sharded_state:
        run_sharded_state(args)
        return
    if args.isdf:
        run_isdf(args)
        return
    if args.sym >= 0 and not args.paper_setting:
        run_sym(args)
        return
    if args.tdc:
        run_tdc(args)
        return

    import torch
    import torch.distributed as dist

    from paper_2310_20103_b200 import gwl, runtime, synth

    rank, local_rank, world = runtime.dist_env()
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    if not os.path.exists(gwl.LIB_PATH):
        if rank == 0:
            from paper_2310_20103_b200 import build
            build.build()
        if world > 1:
            dist.barrier()
    gwl.load_library()

    cfg = synth.CONFIGS[args.config]
    nch, L = pass_shape(args, cfg)
    prob = synth.make_problem(cfg)
    V = prob.V

    def pin(a):
        return torch.from_numpy(np.ascontiguousarray(a)).pin_memory().numpy()

    h = {k: pin(v) for k, v in dict(phi_v=prob.phi_v, phi_c=prob.phi_c, eps_v=prob.eps_v, eps_c=prob.eps_c, V=V,
                                    omega=prob.omega).items()}
    n_idx, m_idx = prob.n_idx[:nch], prob.m_idx[:nch]
    stream = torch.cuda.current_stream()
    flush = torch.empty(L2_FLUSH_BYTES, dtype=torch.uint8, device=dev)
    ev = lambda: torch.cuda.Event(enable_timing=True)  # noqa: E731

    # ---- device-resident arm ----------------------------------------------------------------------
    ctx = gwl.Context(cfg.n_v, cfg.n_c, cfg.n_mu)
    ctx.set_stream(stream.cuda_stream)
    ctx.set_orbitals(h["phi_v"], h["phi_c"])
    ctx.set_energies(h["eps_v"], h["eps_c"])
    ctx.set_kernel(h["V"])
    ctx.set_chains(n_idx, m_idx)
    ctx.set_pointer_mode(1)
    ctx.set_profiling(0)          # no events inside the timed region
    omega_d = torch.from_numpy(prob.omega).to(dev)
    sig_d = torch.empty(nch, cfg.n_omega, 2, dtype=torch.float64, device=dev)
    sum_d = torch.empty(cfg.n_omega, 2, dtype=torch.float64, device=dev)

    def step_device():
        ctx.lanczos(nch, L, cfg.block, 1 if args.reorth else 0, out=None)
        ctx.selfenergy(omega_d, cfg.eta, out=(sig_d, sum_d))

    dmma_peak = gwl.probe_fp64_peak(0)            # also warms the clocks
    dgemm_peak = cublas_dgemm_tflops(dev) if rank == 0 else None
    for _ in range(args.warmup):
        step_device()
    torch.cuda.synchronize()
    sampler = runtime.ClockSampler(local_rank).start()
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    pairs = []
    n0 = ctx.get_launch_count()
    for _ in range(args.steps):
        flush.zero_()
        e0, e1 = ev(), ev()
        e0.record(stream)
        step_device()
        e1.record(stream)
        pairs.append((e0, e1))
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    launches = ctx.get_launch_count() - n0
    elapsed_s = sum(a.elapsed_time(b) for a, b in pairs) * 1e-3
    # Per-kernel durations: the same steps again, immediately, with a CUDA-event pair around every launch
    # (profiling level 2).  Kept out of the timed region above because ~7000 extra events per step cost a few %.
    ctx.set_profiling(2)
    ktimes = {k: [0.0, 0] for k in gwl.KERNEL_CLASSES}
    prof_steps = max(1, min(args.steps, 3))
    prof_pairs = []
    for _ in range(prof_steps):
        flush.zero_()
        e0, e1 = ev(), ev()
        e0.record(stream)
        step_device()
        e1.record(stream)
        prof_pairs.append((e0, e1))
        for k, (ms, cnt) in ctx.get_kernel_times().items():      # synchronises
            ktimes[k][0] += ms
            ktimes[k][1] += cnt
    torch.cuda.synchronize()
    prof_elapsed_s = sum(a.elapsed_time(b) for a, b in prof_pairs) * 1e-3
    ctx.set_profiling(0)
    clocks = sampler.stop()
    units = float(args.steps) * nch * L
    tot_units, max_elapsed = runtime.aggregate_throughput(units, elapsed_s, dev)
    value = tot_units / max_elapsed

    # ---- the dominant kernel against the FP64 tensor roofline ----------------------------------------
    gemm_keys = ("gemm_fwd_KX", "gemm_bwd_KtW", "gemm_V")
    dom = max(gemm_keys, key=lambda k: ktimes[k][0])
    nbl = min(cfg.block, nch)
    blocks = -(-nch // cfg.block)
    flop_launch = {"gemm_fwd_KX": 2.0 * cfg.n_mu * cfg.n_vc * nbl, "gemm_bwd_KtW": 2.0 * cfg.n_mu * cfg.n_vc * nbl,
                   "gemm_V": 2.0 * cfg.n_mu * cfg.n_mu * nbl}
    dom_ms = ktimes[dom][0] / max(ktimes[dom][1], 1)
    achieved = flop_launch[dom] / (dom_ms * 1e-3) / 1e12
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    traffic = None   # dram bytes per launch of that kernel from the committed ncu --set full summary (profiles/traffic.csv)
    try:
        import csv
        for row in csv.DictReader(open(os.path.join(ROOT, "profiles", "traffic.csv"))):
            if int(row["config"]) == args.config and row["kernel_class"] == dom:
                traffic = float(row["dram_bytes_per_launch"])
    except Exception:
        pass
    roofline = {"bound": "tensor", "kernel": f"gemm_tn_dmma<{dom}>", "achieved": achieved, "peak": dmma_peak,
                "unit": "TFLOP/s", "frac": achieved / dmma_peak, "traffic": traffic,
                "peak_source": "live register-resident mma.sync.m8n8k4.f64 (DMMA) issue-rate probe on this GPU "
                               "(gwl_probe_fp64_peak); MEASURED_PEAKS.json has no FP64 entry",
                "peak_cublas_dgemm": dgemm_peak,
                "peak_cublas_dgemm_how": "torch.matmul float64 8192^3, best of 3, same process (context: what the "
                                         "vendor library reaches on the same pipe)",
                "peak_from_bf16_ratio": (peaks.get("bf16_tflops", 0) * 37.0 / 2250.0) or None,
                "flop_per_launch": flop_launch[dom], "ms_per_launch": dom_ms, "launches_timed": ktimes[dom][1],
                "timed_how": f"CUDA-event pair around every launch on the library's stream, {prof_steps} extra steps "
                             "run right after the timed region (events inside it would perturb the step time)"}
    step_ms = 1e3 * elapsed_s / args.steps
    share = {k: round(v[0] / (1e3 * prof_elapsed_s), 4) for k, v in ktimes.items() if v[1]}
    # block products inside the Lanczos loop only: S1 launches one V.T and one K^T.W per block on top of the L steps
    n_mv = prof_steps * blocks * L
    per = {k: ktimes[k][0] / max(ktimes[k][1], 1) for k in ("gemm_fwd_KX", "gemm_V", "gemm_bwd_KtW")}
    # split-K reductions: two per product inside the loop (K.X, V.T), one per block in S1 (V.T)
    red_ms = 2.0 * ktimes["splitk_reduce"][0] / (prof_steps * blocks * (2 * L + 1))
    mv_ms = per["gemm_fwd_KX"] + per["gemm_V"] + per["gemm_bwd_KtW"] + red_ms
    fpv = cfg.flop_per_vector() * nbl
    matvec = {"tflops": fpv / (mv_ms * 1e-3) / 1e12, "ms_per_block_matvec": mv_ms,
              "frac_of_dmma_peak": fpv / (mv_ms * 1e-3) / 1e12 / dmma_peak,
              "flop_model": "(4 N_mu N_vc + 2 N_mu^2) B", "block_products_timed": n_mv,
              "how": "mean launch duration of K.X + V.T + K^T.W (+ split-K reductions per product)"}

    # ---- the block product alone, through its own C-ABI call (gwl_casida_matvec, device pointers), back to back ----------
    # (the per-launch sum above is taken with an event pair around every launch, which breaks the overlap of a kernel's
    # prologue with its predecessor's tail; this is the same product as a user calls it, launch gaps included)
    xb = torch.randn(nbl, cfg.n_v, cfg.n_c, dtype=torch.float64, device=dev)
    yb = torch.empty_like(xb)
    mv_reps = max(3, min(200, int(0.5 / max(mv_ms * 1e-3, 1e-6))))
    for _ in range(2):
        ctx.casida_matvec(xb, yb)
    torch.cuda.synchronize()
    m0, m1 = ev(), ev()
    m0.record(stream)
    for _ in range(mv_reps):
        ctx.casida_matvec(xb, yb)
    m1.record(stream)
    torch.cuda.synchronize()
    abi_ms = m0.elapsed_time(m1) / mv_reps
    matvec["abi_call"] = {"ms_per_block_matvec": abi_ms, "tflops": fpv / (abi_ms * 1e-3) / 1e12,
                          "frac_of_dmma_peak": fpv / (abi_ms * 1e-3) / 1e12 / dmma_peak, "reps": mv_reps,
                          "how": "gwl_casida_matvec(block) in device-pointer mode, back-to-back calls between two CUDA "
                                 "events; includes the sqrt(Delta) prescale kernel and every launch gap"}
    del xb, yb

    # ---- end-to-end arm: host buffers through the C ABI --------------------------------------------------
    e2e = None
    if not args.no_e2e:
        hctx = gwl.Context(cfg.n_v, cfg.n_c, cfg.n_mu)
        hctx.set_stream(stream.cuda_stream)
        hctx.set_profiling(0)

        def step_host():
            hctx.set_orbitals(h["phi_v"], h["phi_c"])
            hctx.set_energies(h["eps_v"], h["eps_c"])
            hctx.set_kernel(h["V"])
            hctx.set_chains(n_idx, m_idx)
            out = hctx.lanczos(nch, L, cfg.block, 0)
            sig = hctx.selfenergy(h["omega"], cfg.eta, nch)
            return out, sig

        for _ in range(min(args.warmup, 2)):
            step_host()
        ke = max(1, args.steps)
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        hp = []
        for _ in range(ke):
            flush.zero_()
            e0, e1 = ev(), ev()
            e0.record(stream)
            step_host()
            e1.record(stream)
            hp.append((e0, e1))
        torch.cuda.synchronize()
        he = sum(a.elapsed_time(b) for a, b in hp) * 1e-3
        hu, ht = runtime.aggregate_throughput(float(ke) * nch * L, he, dev)
        h2d = sum(h[k].nbytes for k in ("phi_v", "phi_c", "eps_v", "eps_c", "V", "omega")) + 2 * 4 * nch + 12 * nch
        d2h = nch * L * 16 + nch * 12 + nch * cfg.n_omega * 16 + cfg.n_omega * 16
        e2e = {"value": hu / ht, "unit": UNIT, "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
               "steps": ke, "ms_per_step": 1e3 * he / ke, "ms_each": [round(a.elapsed_time(b), 3) for a, b in hp]}
        hctx.close()

    if rank == 0:
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": step_ms, "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": workload_config(cfg, world, L, nch),
                "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline, "matvec": matvec,
                "kernel_time_share": share}
        if args.lanczos_steps or args.chains:
            line["note"] = "chains / lanczos_steps overridden: profiling run, not a bench value"
        if args.reorth:
            line["note"] = "full reorthogonalisation on: not the bench workload"
            line["config"]["mode"] = "direct (Op = C), reorth on (CGS2)"
            rt = ktimes["reorth"]
            # CGS2 at step k reads the k+1 basis vectors twice per pass (dots, apply), two passes
            nbytes = prof_steps * 4.0 * 8.0 * cfg.n_vc * nch * (L * (L + 1) / 2.0)
            line["reorth"] = {"ms_per_pass_of_L_steps": rt[0] / prof_steps, "algorithmic_GBps": nbytes / (rt[0] * 1e-3) / 1e9}
        if world == 1 and not args.no_cpu_baseline:
            line["cpu_baseline"] = cpu_baseline(prob, nch, L)
        print(json.dumps(line), flush=True)
    ctx.close()
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
