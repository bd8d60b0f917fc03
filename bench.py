#!/usr/bin/env python
"""bench.py -- measures the loop-integral hot path on B200 (contract: see DESIGN.md "Measurement").

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--no-others] [--no-cpu-baseline]
                    [--full] [--report FILE] [--issue-model]

--gpus N > 1: one rank per GPU, weak scaling (64 external momenta per rank, no data-path collective).  Either start the
ranks yourself (`python -m torch.distributed.run --nnodes=1 --nproc-per-node N --master-addr 127.0.0.1 --master-port P
bench.py --gpus N ...`) or run `python bench.py --gpus N ...` plainly: without a launcher environment the script starts
the N ranks itself, and it refuses to run if fewer than N devices are visible.  Rank 0 prints the line.

A step is one pass of the whole hot path (S1..S6) over one batch: BASELINE.json configs[4], the
finite-T momentum-dependent loop (64 p x 16 Matsubara indices x 512 field points = 524 288 integrals,
52 992 quadrature nodes each), the largest single-GPU configuration.  `value` = nominal integrand
evaluations per second with inputs resident in HBM; `e2e` = the same through the host-buffer C-ABI
call (node generation + H2D + kernel + D2H in the timed region).  One JSON line on stdout.

--full compares ALL outputs of the workload with the CPU oracle (about 2.5 minutes of host time on 16 cores) instead
of the bounded sample of the default cpu_baseline leg; --report FILE also writes that comparison as JSON to FILE.
The process exits 1 (after printing the line) if the comparison breaks a bar of DESIGN.md "Parity bar".
"""
import argparse
import json
import math
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "fp64_integrand_evals_per_s"
UNIT = "evals/s"
WORKLOAD = "cfg4_matsubara3d: 64 p x 16 j x 512 field points, 23 Matsubara terms x 96 q x 24 cos nodes, FP64"

# FP64 roofline denominator: 148 SMs x 64 FP64 lanes x 2 flop/DFMA x 1.965 GHz
FP64_LANES_PER_SM = 64
# the committed `ncu --set full` capture of the bench kernel on this workload: roofline.traffic is read from it
NCU_CAPTURE = os.path.join("profiles", "r3_bench_kernel.md")


def ncu_dram_bytes_per_launch():
    """dram__bytes_read.sum + dram__bytes_write.sum of the moment kernel, per launch, from the committed ncu summary
    (a run under ncu is never a bench run, so the number cannot be measured here); None if the file is missing."""
    unit = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}
    try:
        tot, seen = 0.0, set()
        for ln in open(os.path.join(ROOT, NCU_CAPTURE)):
            f = [t.strip() for t in ln.strip().strip("|").split("|")]
            if len(f) == 3 and f[0] in ("dram__bytes_read.sum", "dram__bytes_write.sum") and f[0] not in seen:
                seen.add(f[0])
                tot += float(f[1]) * unit[f[2]]
        return int(round(tot)) if len(seen) == 2 else None
    except (OSError, KeyError, ValueError):
        return None


def cfg4_counts(c, rules):
    n_p, n_j, n_f = c["pext"].size, c["n_jext"], c["m2psi"].size
    n_out = n_p * n_j * n_f
    n_terms = 2 * c["n_max"] + 1
    nq, nc = rules["q"][0].size, rules["c"][0].size
    evals = n_out * n_terms * nq * nc
    # algorithmic FP64 work of the moment factorisation, per (p, radial node, field point):
    #   (n_j + n_max) nc x 7   angular moments of the boson line   (DADD, 3 DFMA reciprocal, and per symmetric node
    #                          pair (c, -c) 2 DADD + 4 DFMA: M_b += w c^b (r+ +- r-))
    # + (n_max + 1) x 5        fermion line G_psi^2                (DADD, 3 DFMA, DMUL)
    # + n_j n_terms x 5        acc_j += H (beta' . M)              (DMUL, 3 DFMA, DFMA)
    # flops = DFMA-slot equivalents (2 per instruction); strict = FMA 2, add/mul 1.
    rows = n_j + c["n_max"]
    per_pif = rows * nc * 7 + (c["n_max"] + 1) * 5 + n_j * n_terms * 5
    per_pif_strict = rows * nc * 12 + (c["n_max"] + 1) * 8 + n_j * n_terms * 9
    units = n_p * nq * n_f
    return n_out, evals, (2.0 * units * per_pif, float(units * per_pif_strict))


def cfg4_reciprocals(c, rules):
    """Reciprocals the moment factorisation executes per step: per (p, radial node, field point) one per boson-line row
    and cos node and one per fermion-line term (the nominal count `evals` has one propagator pair per (n, q, c) node of
    every output; the factorisation shares the boson-line reciprocals over the (j, n) pairs with equal |j - n|)."""
    nq, nc = rules["q"][0].size, rules["c"][0].size
    return c["pext"].size * nq * c["m2psi"].size * ((c["n_jext"] + c["n_max"]) * nc + c["n_max"] + 1)


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 20 ms under load.  The timed region of a default run lasts tens of
    milliseconds -- shorter than nvidia-smi takes to start -- so the sampler is started before an untimed pre-load phase of the
    same steps (0.3 s) that runs straight into the timed steps; the samples cover pre-load + timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None
        self.index = index

    def start(self):
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                       "--format=csv,noheader,nounits", "-lms", "20"], stdout=self.f,
                                      stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None

    def stop(self):
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.p.terminate()
        self.p.wait()
        self.f.flush()
        self.f.seek(0)
        rows = [r.split(",") for r in self.f.read().strip().splitlines() if r.count(",") >= 6]
        os.unlink(self.f.name)
        if not rows:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        sm = sorted(float(r[0]) for r in rows)
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [nm for i, nm in enumerate(names) if any("Active" in r[3 + i] and "Not" not in r[3 + i] for r in rows)]
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": float(rows[0][1]), "samples": len(rows),
                "window": "untimed pre-load of the same steps (0.3 s) + the timed region, sampled every 20 ms",
                "power_w_max": max(float(r[2]) for r in rows), "reasons": reasons}


def run_reference(args):
    """--impl reference: the CPU oracle as it stands on the host cores, a bounded sample per step."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    import oracle
    from oracle.harness import oracle_run
    from paper_2412_13043_b200 import inputs
    c = inputs.config4()
    R = inputs.make_rules(c, oracle.gl_rule)
    n_out, evals, _ = cfg4_counts(c, R)
    stride = 512
    sel = np.arange(0, n_out, stride)                       # 1024 outputs per step
    per_out = evals // n_out
    for _ in range(args.warmup):
        oracle_run(c, R, sel=sel[:64])
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle_run(c, R, sel=sel)
    dt = (time.perf_counter() - t0) / args.steps
    val = sel.size * per_out / dt
    cores = oracle.num_threads()
    sample = "%d of %d outputs per step (every %dth), %d nodes each" % (sel.size, n_out, stride, per_out)
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": WORKLOAD, "sample": sample},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "integrals_per_s": sel.size / dt}
    print(json.dumps(line))
    return 0


def alu_roofline(alg_instr, alg_flops_strict, ms, peak, what):
    """roofline block of an FP64-pipe-bound kernel.  `achieved` / `frac`: algorithmic flops counted strictly (FMA 2,
    add / mul 1) against the nominal FP64 peak in TFLOP/s.  `fp64_pipe_utilisation`: algorithmic FP64
    instructions / the pipe's issue slots in the measured time (a DADD or DMUL holds the pipe as long as a DFMA) -- the
    figure ncu's sm__pipe_fp64_cycles_active measures, and the one the >= 50 % target of SURVEY 8(d) is worded on."""
    strict = alg_flops_strict / (ms * 1e-3) * 1e-12
    slots = 2.0 * alg_instr / (ms * 1e-3) * 1e-12
    return {"bound": "alu", "achieved": strict, "peak": peak, "unit": "TFLOP/s", "frac": strict / peak,
            "achieved_kind": "algorithmic flops, FMA = 2, add / mul = 1 (" + what + ")",
            "fp64_pipe_utilisation": slots / peak, "alg_fp64_instr_per_launch": alg_instr,
            "alg_fp64_instr_per_s": alg_instr / (ms * 1e-3), "alg_flops_per_launch": alg_flops_strict}


def time_other_configs(torch, B, inputs, make_rules, peak, iters=5):
    """Device-resident timings of configs 0-3 (context for the flagship loop4d kernels; not the bench line)."""
    out = {}

    def timeit(fn, n=iters, reps=1):
        """median over n timings of `reps` back-to-back calls (reps > 1 keeps the host launch latency of a
        tens-of-microseconds kernel out of the device time); ms per call"""
        for _ in range(2):
            fn()
        torch.cuda.synchronize()
        ts = []
        for _ in range(n):
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            for _ in range(reps):
                fn()
            b.record()
            b.synchronize()
            ts.append(a.elapsed_time(b) / reps)
        return float(np.median(ts))

    up = lambda a: torch.as_tensor(np.ascontiguousarray(a)).cuda()
    # cfg0 / cfg1
    for name, cs in (("cfg0", [inputs.config0()]), ("cfg1", [inputs.config1(T) for T in inputs.CONFIG1_TEMPERATURES])):
        calls, evals, integrals = [], 0, 0
        for c in cs:
            R = make_rules(c, B.dfrg_quad_nodes)
            rq = (up(R["q"][0]), up(R["q"][1]))
            rho, u, du = up(c["rho"]), up(c["u"]), up(c["du"])
            flow = torch.empty_like(rho)
            calls.append((c, rq, rho, u, du, flow))
            terms = (2 * c["n_max"] + 1) if c["T"] > 0 else 1
            evals += 2 * rho.numel() * terms * rq[0].numel()
            integrals += 2 * rho.numel()

        def fn():
            for c, rq, rho, u, du, flow in calls:
                B.dfrg_integrate_lpa(c["d"], c["T"], c["n_max"], c["reg_arg4d"], c["N"], c["prefactor"], c["reg_kind"],
                                     c["reg_order"], c["k"], rq, rho, u, du, flow)
        ms = timeit(fn, reps=20)
        out[name] = {"ms": ms, "evals_per_s": evals / ms * 1e3, "integrals_per_s": integrals / ms * 1e3,
                     "launches": len(calls)}
        if name == "cfg1":
            # the four temperatures of config 1 captured once into a CUDA graph and replayed (no host work per call)
            fn()
            torch.cuda.synchronize()
            graph = torch.cuda.CUDAGraph()
            with torch.cuda.graph(graph):
                fn()
            msg = timeit(graph.replay, reps=20)
            out["cfg1_cuda_graph"] = {"ms": msg, "evals_per_s": evals / msg * 1e3, "integrals_per_s": integrals / msg * 1e3,
                                      "launches": len(calls)}
            # ... and as ONE launch through dfrg_integrate_lpa_batch (grid.y = temperature)
            c0 = calls[0][0]
            fb = torch.empty(len(calls), calls[0][2].numel(), dtype=torch.float64, device="cuda")
            msb = timeit(lambda: B.dfrg_integrate_lpa_batch(c0["d"], [cc[0]["T"] for cc in calls], [cc[0]["n_max"] for cc in calls],
                                                            c0["reg_arg4d"], c0["N"], c0["prefactor"], c0["reg_kind"],
                                                            c0["reg_order"], c0["k"], calls[0][1], calls[0][2], calls[0][3],
                                                            calls[0][4], fb), reps=20)
            assert all(torch.equal(fb[t_], calls[t_][5]) for t_ in range(len(calls)))
            out["cfg1_batched"] = {"ms": msb, "evals_per_s": evals / msb * 1e3, "integrals_per_s": integrals / msb * 1e3,
                                   "launches": 1}
    # cfg2
    c = inputs.config2()
    R = make_rules(c, B.dfrg_quad_nodes)
    rq, rc = (up(R["q"][0]), up(R["q"][1])), (up(R["c"][0]), up(R["c"][1]))
    Z, coef, m2, pext = up(c["Z"]), up(c["coef"]), up(c["m2"]), up(c["pext"])
    o2 = torch.empty(pext.numel(), m2.numel(), dtype=torch.float64, device="cuda")
    f2 = lambda: B.dfrg_integrate_loop4d(B.LOOP_TWOPOINT, c["prefactor"], c["reg_kind"], c["reg_order"], c["k"],
                                         rq, rc, None, None, (Z,), c["lnq_lo"], c["lnq_hi"], c["interp"], coef, m2, pext, o2)
    ms_eager = timeit(f2, reps=20)
    # The call is two kernels of ~30 + 3 us: issued one by one from Python the stream runs dry between calls (the host needs
    # ~40 us per call), so the device time is taken from a CUDA graph of 20 calls replayed back to back.
    torch.cuda.synchronize()
    g2 = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g2):
        for _ in range(20):
            f2()
    ms = timeit(g2.replay, reps=1) / 20.0
    ev = o2.numel() * rq[0].numel() * rc[0].numel()
    # per (p, q, field point) one pair inversion per two cos nodes (4.5 instr per node: DADD, 3 DFMA
    # Newton, 1/2 DMUL + ... ) and 5.5 per radial node; strict flops: 8 per node + 10 per radial node
    n_pqf = o2.numel() * rq[0].numel()
    out["cfg2"] = {"ms": ms, "ms_kind": "device time per call: CUDA graph of 20 calls replayed (main + fix-up kernel)",
                   "ms_eager_python": ms_eager, "evals_per_s": ev / ms * 1e3, "integrals_per_s": o2.numel() / ms * 1e3,
                   "launches": 2,
                   "roofline": alu_roofline(n_pqf * (4.5 * rc[0].numel() + 5.5), n_pqf * (8.0 * rc[0].numel() + 10.0), ms,
                                            peak, "tp_main_kernel: 4.5 FP64 instr per (p, q, c, field point) + 5.5 per "
                                                  "(p, q, field point)")}
    # cfg3
    c = inputs.config3()
    R = make_rules(c, B.dfrg_quad_nodes)
    rr = {k_: (up(v[0]), up(v[1])) for k_, v in R.items()}
    tabs = (up(c["ZA"]), up(c["Zc"]), up(c["L3"]))
    coef, ext = up(c["coef"]), up(c["ext"])
    o3 = torch.empty(ext.shape[0], dtype=torch.float64, device="cuda")
    ms = timeit(lambda: B.dfrg_integrate_loop4d(B.LOOP_THREEPOINT, c["prefactor"], c["reg_kind"], c["reg_order"],
                                                c["k"], rr["q"], rr["c1"], rr["c2"], rr["phi"], tabs, c["lnq_lo"],
                                                c["lnq_hi"], c["interp"], coef, None, ext, o3,
                                                ext_outer=c["ext_outer"]), n=3)
    uniq = o3.numel() * rr["q"][0].numel() * rr["c1"][0].numel() * rr["c2"][0].numel()
    # 17 FP64 instr per unique node (a, r, q, c1, c2); 45 per shared node (r, q, c1, c2) of phase 1
    # (G_A(s_b) and its vertex); 85 per (|p1|, q, c1) of the pre-pass; 2 per row.  strict: 15 of the 17 are FMAs.
    G = c["ext_outer"]
    S = o3.numel() // G
    npairs, n2 = rr["q"][0].numel() * rr["c1"][0].numel(), rr["c2"][0].numel()
    alg3 = uniq * 17.0 + S * npairs * n2 * 45.0 + G * npairs * 85.0 + o3.numel() * npairs * 2.0
    alg3s = uniq * 32.0 + S * npairs * n2 * 80.0 + G * npairs * 160.0 + o3.numel() * npairs * 2.0
    out["cfg3"] = {"ms": ms, "unique_evals_per_s": uniq / ms * 1e3,
                   "nominal_evals_per_s": uniq * rr["phi"][0].numel() / ms * 1e3,
                   "integrals_per_s": o3.numel() / ms * 1e3,
                   "launches": 4,   # product-grid path: pre-pass, main, fix-up, and the general kernel returning at once
                   "roofline": alu_roofline(alg3, alg3s, ms, peak, "t3g_main_kernel (+ pre-pass and fix-up, timed "
                                            "together): 17 FP64 instr per unique node, 45 per shared node, 85 per "
                                            "pre-pass entry")}
    # cfg5 (four-point box, genuine three-angle kinematics + ghost loop; SURVEY 8(f) item 3 -- not a BASELINE config)
    c = inputs.config5()
    R = make_rules(c, B.dfrg_quad_nodes)
    rr = {k_: (up(v[0]), up(v[1])) for k_, v in R.items()}
    tabs = (up(c["ZA"]), up(c["Zc"]), up(c["L3"]))
    coef, ext = up(c["coef"]), up(c["ext"])
    o5 = torch.empty(ext.shape[0], dtype=torch.float64, device="cuda")
    ms = timeit(lambda: B.dfrg_integrate_loop4d(B.LOOP_FOURPOINT, c["prefactor"], c["reg_kind"], c["reg_order"],
                                                c["k"], rr["q"], rr["c1"], rr["c2"], rr["phi"], tabs, c["lnq_lo"],
                                                c["lnq_hi"], c["interp"], coef, None, ext, o5), n=3)
    ev = o5.numel() * rr["q"][0].numel() * rr["c1"][0].numel() * rr["c2"][0].numel() * rr["phi"][0].numel()
    out["cfg5_fourpoint"] = {"ms": ms, "evals_per_s": ev / ms * 1e3, "integrals_per_s": o5.numel() / ms * 1e3,
                             "launches": 2}
    # cfg6 (three-point with the paper-shaped 96 x 8 x 7 vertex table in shared memory)
    c = inputs.config6()
    R = make_rules(c, B.dfrg_quad_nodes)
    rr = {k_: (up(v[0]), up(v[1])) for k_, v in R.items()}
    coef, ext, ZA, v3 = up(c["coef"]), up(c["ext"]), up(c["ZA"]), up(c["v3"])
    o6 = torch.empty(ext.shape[0], dtype=torch.float64, device="cuda")
    ms = timeit(lambda: B.dfrg_integrate_loop4d(B.LOOP_THREEPOINT_TAB3D, c["prefactor"], c["reg_kind"], c["reg_order"],
                                                c["k"], rr["q"], rr["c1"], rr["c2"], rr["phi"], (ZA,), c["lnq_lo"],
                                                c["lnq_hi"], c["interp"], coef, None, ext, o6,
                                                tab3d=(v3, c["lo3"], c["hi3"], c["log3"]),
                                                ext_outer=c["ext_outer"]), n=3)
    uniq = o6.numel() * rr["q"][0].numel() * rr["c1"][0].numel() * rr["c2"][0].numel()
    out["cfg6_threepoint_tab3d"] = {"ms": ms, "unique_evals_per_s": uniq / ms * 1e3,
                                    "table_lookups_per_s": uniq * (2 + 1.0 / rr["c2"][0].numel()) / ms * 1e3,
                                    "integrals_per_s": o6.numel() / ms * 1e3, "launches": 4}
    # cfg4 with both mass derivatives (three passes of the moment kernel: value, d/dm2_psi, d/dm2_phi)
    c = inputs.config4()
    R = make_rules(c, B.dfrg_quad_nodes)
    rq, rc = (up(R["q"][0]), up(R["q"][1])), (up(R["c"][0]), up(R["c"][1]))
    Zpsi, Zphi, coef = up(c["Zpsi"]), up(c["Zphi"]), up(c["coef"])
    m2psi, m2phi, pext = up(c["m2psi"]), up(c["m2phi"]), up(c["pext"])
    o4 = [torch.empty(pext.numel(), c["n_jext"], m2psi.numel(), dtype=torch.float64, device="cuda") for _ in range(3)]
    ms = timeit(lambda: B.dfrg_integrate_matsubara3d(c["T"], c["n_max"], c["prefactor"], c["reg_kind"], c["reg_order"],
                                                     c["k"], rq, rc, Zpsi, Zphi, c["lnq_lo"], c["lnq_hi"], c["interp"],
                                                     coef, m2psi, m2phi, pext, c["n_jext"], o4[0], dout_dm2_psi=o4[1],
                                                     dout_dm2_phi=o4[2]), n=3)
    o_im = torch.empty_like(o4[0])
    ms_mu = timeit(lambda: B.dfrg_integrate_matsubara3d(c["T"], c["n_max"], c["prefactor"], c["reg_kind"], c["reg_order"],
                                                        c["k"], rq, rc, Zpsi, Zphi, c["lnq_lo"], c["lnq_hi"], c["interp"],
                                                        coef, m2psi, m2phi, pext, c["n_jext"], o4[0], reg_arg4d=0, mu=0.3,
                                                        out_im=o_im), n=3)
    ev4 = o4[0].numel() * (2 * c["n_max"] + 1) * rq[0].numel() * rc[0].numel()
    out["cfg4_chemical_potential"] = {"ms": ms_mu, "evals_per_s": ev4 / ms_mu * 1e3,
                                      "integrals_per_s": o4[0].numel() / ms_mu * 1e3, "launches": 6,
                                      "note": "mu = 0.3 k, spatial regulators, complex result (SURVEY 8(f) item 4)"}
    out["cfg4_with_mass_derivatives"] = {"ms": ms, "integrals_and_derivatives_per_s": 3 * o4[0].numel() / ms * 1e3,
                                         "launches": 8}
    return out


def rank_env(n_gpus_arg):
    """(rank, world, local rank) of this process from the launcher's environment (torchrun sets RANK / WORLD_SIZE /
    LOCAL_RANK); a plain single-process run is rank 0 of 1.  --gpus must agree with the world size."""
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", str(rank)))
    if not (0 <= rank < world):
        raise SystemExit("bench.py: RANK %d outside WORLD_SIZE %d" % (rank, world))
    if n_gpus_arg != world:
        raise SystemExit("bench.py: --gpus %d but the launcher started %d rank(s)" % (n_gpus_arg, world))
    return rank, world, local


def rank_workload(inputs, shard_bounds, world, rank):
    """This rank's share of the global batch.  Weak scaling: the global batch has 64 x world external momenta on the same
    log range; rank r integrates its contiguous block; no data-path collective."""
    c = inputs.config4(n_p=64 * world)
    lo_p, hi_p = shard_bounds(c["pext"].size, world, rank)
    c["pext_global_range"] = (lo_p, hi_p)
    c["pext"] = np.ascontiguousarray(c["pext"][lo_p:hi_p])
    return c


def max_over_ranks(x, dist, device):
    """MAX over ranks of a per-rank time (the job is as slow as its slowest rank); dist = None: single process."""
    if dist is None:
        return float(x)
    import torch
    t = torch.tensor([float(x)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_rate(world, units_per_rank, ms):
    """units per second over ALL ranks: every rank processed units_per_rank in the (max-over-ranks) time ms."""
    return world * units_per_rank / (ms * 1e-3)


def launch_ranks(n, argv):
    """`python bench.py --gpus N` with N > 1 and no launcher environment: starts N ranks (one per GPU) of this script under
    torch.distributed.run on 127.0.0.1 and returns its exit code.  Rank 0 prints the JSON line.  NCCL's communicator set-up
    lines go to stderr (NCCL_DEBUG=INFO, INIT subsystem) unless the caller has set NCCL_DEBUG."""
    import socket
    import torch
    have = torch.cuda.device_count()
    if have < n:
        raise SystemExit("bench.py --gpus %d: only %d CUDA device(s) visible; refusing to run fewer ranks than asked" % (n, have))
    with socket.socket() as sock:
        sock.bind(("127.0.0.1", 0))
        port = sock.getsockname()[1]
    env = dict(os.environ)
    if "NCCL_DEBUG" not in env:
        env.update(NCCL_DEBUG="INFO", NCCL_DEBUG_SUBSYS="INIT", NCCL_DEBUG_FILE="/dev/stderr")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(n), "--master-addr",
           "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + list(argv)
    return subprocess.call(cmd, env=env)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-others", action="store_true", help="skip the context timings of configs 0-3")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--full", action="store_true", help="compare every output of the workload with the CPU oracle")
    ap.add_argument("--report", default=None, help="write the oracle comparison as JSON to this file")
    ap.add_argument("--issue-model", action="store_true",
                    help="also run the FP64 issue-model probe (DESIGN.md section 7) and add it to the roofline block")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        return run_reference(args)
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        return launch_ranks(args.gpus, sys.argv[1:])         # `python bench.py --gpus N`: start the N ranks ourselves

    import torch
    from paper_2412_13043_b200 import binding as B
    from paper_2412_13043_b200 import inputs
    from paper_2412_13043_b200.inputs import make_rules
    from paper_2412_13043_b200.shard import shard_bounds

    rank, world, local = rank_env(args.gpus)
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback")
    if torch.cuda.device_count() <= local:
        raise SystemExit("bench.py: rank %d wants cuda:%d but only %d device(s) are visible" %
                         (rank, local, torch.cuda.device_count()))
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    B.lib()  # fail loudly if libdfrg.so is missing

    # ---- workload (weak scaling: the global batch has 64 x N external momenta on the same log range; every
    # rank integrates its contiguous block of 64; no data-path collective) ----
    c = rank_workload(inputs, shard_bounds, world, rank)
    t_s1 = time.perf_counter()
    R = make_rules(c, B.dfrg_quad_nodes)                     # S1, host
    t_s1 = time.perf_counter() - t_s1
    n_out, evals, (flops, flops_strict) = cfg4_counts(c, R)
    up = lambda a: torch.as_tensor(np.ascontiguousarray(a)).cuda()
    rq, rc = (up(R["q"][0]), up(R["q"][1])), (up(R["c"][0]), up(R["c"][1]))
    Zpsi, Zphi, coef = up(c["Zpsi"]), up(c["Zphi"]), up(c["coef"])
    m2psi, m2phi, pext = up(c["m2psi"]), up(c["m2phi"]), up(c["pext"])
    out = torch.empty(pext.numel(), c["n_jext"], m2psi.numel(), dtype=torch.float64, device="cuda")
    flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device="cuda")   # > 126 MB L2

    def step():
        B.dfrg_integrate_matsubara3d(c["T"], c["n_max"], c["prefactor"], c["reg_kind"], c["reg_order"], c["k"], rq, rc,
                                     Zpsi, Zphi, c["lnq_lo"], c["lnq_hi"], c["interp"], coef, m2psi, m2phi, pext,
                                     c["n_jext"], out)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- FP64 peak probe (register-only DFMA chains), before the timed region ----
    sink = torch.zeros(8, dtype=torch.float64, device="cuda")
    from paper_2412_13043_b200 import probe
    probe.fp64_peak(2000, 2, sink)
    torch.cuda.synchronize()
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record()
    probe_flops = probe.fp64_peak(40000, 2, sink)
    b.record()
    b.synchronize()
    probe_tflops = probe_flops / (a.elapsed_time(b) * 1e-3) * 1e-12
    issue_model = probe.fp64_issue_model(sink) if args.issue_model else None   # 8 DFMA + K other instructions: DESIGN.md section 7

    for _ in range(args.warmup):
        step()
    barrier()
    sampler = ClockSampler(local)
    sampler.start()
    t_pre = time.perf_counter()
    while time.perf_counter() - t_pre < 0.3:                  # untimed pre-load: the GPU is under the same load when the
        for _ in range(8):                                     # timed steps start, and the clock sampler is up
            step()
        torch.cuda.synchronize()
    evs = []
    barrier()
    t_wall = time.perf_counter()
    for _ in range(args.steps):
        flush.fill_(1)                                        # L2 flush between timed iterations (not timed)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        step()
        e1.record()
        evs.append((e0, e1))
    barrier()
    t_wall = time.perf_counter() - t_wall
    clocks = sampler.stop()
    ms_local = sum(e0.elapsed_time(e1) for e0, e1 in evs) / args.steps
    ms = max_over_ranks(ms_local, dist, "cuda")
    value = whole_job_rate(world, evals, ms)

    # ---- e2e: host buffers through the C ABI, S1 + H2D + kernel + D2H inside the timed region ----
    pin = lambda a: torch.as_tensor(np.ascontiguousarray(a)).pin_memory()
    h = {k_: pin(c[k_]) for k_ in ("Zpsi", "Zphi", "coef", "m2psi", "m2phi", "pext")}
    h_out = torch.empty(out.shape, dtype=torch.float64).pin_memory()
    hx = {ax: (torch.empty(R[ax][0].size, dtype=torch.float64).pin_memory(),
               torch.empty(R[ax][0].size, dtype=torch.float64).pin_memory()) for ax in ("q", "c")}

    def e2e_step():
        for ax in ("q", "c"):                                  # S1 on the host, into pinned buffers
            n_, a_, b_ = c["rule_" + ax]
            rc_ = B.lib().dfrg_quad_nodes(0, n_, a_, b_, hx[ax][0].data_ptr(), hx[ax][1].data_ptr())
            assert rc_ == 0
        B.dfrg_integrate_matsubara3d_host(c["T"], c["n_max"], c["prefactor"], c["reg_kind"], c["reg_order"], c["k"],
                                          hx["q"], hx["c"], h["Zpsi"], h["Zphi"], c["lnq_lo"], c["lnq_hi"], c["interp"],
                                          h["coef"], h["m2psi"], h["m2phi"], h["pext"], c["n_jext"], h_out)
    e2e_steps = max(3, min(args.steps, 10))
    e2e_step()
    barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        e2e_step()
    barrier()
    e2e_s = (time.perf_counter() - t0) / e2e_steps
    e2e_s = max_over_ranks(e2e_s, dist, "cuda")
    rows_psi, rows_phi = c["n_max"] + 1, c["n_jext"] + c["n_max"]
    h2d = 8 * (2 * (R["q"][0].size + R["c"][0].size) + (rows_psi + rows_phi) * c["Zpsi"].shape[1] + 20 +
               2 * c["m2psi"].size + c["pext"].size)
    d2h = 8 * n_out
    assert torch.equal(h_out.cuda(), out), "host and device entry points disagree"

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return 0

    sm_max_mhz = clocks.get("sm_max_mhz") or 1965.0
    sms = torch.cuda.get_device_properties(local).multi_processor_count
    peak = sms * FP64_LANES_PER_SM * 2 * sm_max_mhz * 1e6 * 1e-12          # TFLOP/s at max clock
    roof = alu_roofline(flops / 2.0, flops_strict, ms_local, peak,
                        "moment factorisation: 7 FP64 instr per (boson row, cos node), 5 per fermion term, 5 per (j, n), "
                        "each per (p, radial node, field point)")
    alg_bytes = 8 * c["pext"].size * rows_phi * R["q"][0].size * R["c"][0].size
    roof.update({
        "kernel": "mats3d_moment_kernel (+ the two pre-pass kernels and the fix-up kernel, timed together)",
        "traffic": ncu_dram_bytes_per_launch() if world == 1 else None,
        "traffic_kind": "MOMENT KERNEL ONLY: dram__bytes_read.sum + dram__bytes_write.sum of mats3d_moment_kernel per launch, a "
                        "constant read at run time from the committed ncu --set full capture of this workload (" + NCU_CAPTURE +
                        "), not measured by this run; its algorithmic bytes are the D0phi chunks [p][27 rows][q][c], read once",
        "alg_bytes_per_launch": alg_bytes,
        "alg_bytes_per_step": 2 * alg_bytes + 8 * n_out,
        "alg_bytes_per_step_kind": "the pre-pass writes the D0phi table, the moment kernel reads it once, the fix-up writes the "
                                   "outputs (partial sums and the small tables stay in L2): about 68 MB, 1 % of the HBM "
                                   "bandwidth at this step time",
        "alg_fp64_instr_per_nominal_eval": flops / 2.0 / evals,
        "peak_kind": "nominal FP64: %d SMs x %d lanes x 2 x %.0f MHz (MEASURED_PEAKS.json has no FP64 "
                     "entry)" % (sms, FP64_LANES_PER_SM, sm_max_mhz),
        "peak_probe_tflops": probe_tflops, "frac_of_probe": roof["achieved"] / probe_tflops})
    if issue_model is not None:
        roof["issue_model_probe"] = dict(issue_model, kind="time of 8 DFMA chains + K instructions of another pipe per 8 DFMA "
                                         "(integer add, I2F.F64, LDS.128) relative to K = 0; integer-add ratios "
                                         "(16 + K)/16 would mean an FP64 instruction holds the issue port for 2 "
                                         "cycles, ratios of 1 that other instructions issue in its shadow")
    n_recip = cfg4_reciprocals(c, R)
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic",
            "value_kind": "NOMINAL integrand evaluations (one per output and (n, q, c) node, the count BASELINE.json's metric "
                          "names); the executed work after the exact moment factorisation is in executed_reciprocals_per_s "
                          "and alg_fp64_instr_per_s",
            "executed_reciprocals_per_s": whole_job_rate(world, n_recip, ms),
            "alg_fp64_instr_per_s": whole_job_rate(world, flops / 2.0, ms),
            "config": {"workload": WORKLOAD, "l2": "flushed between timed steps (256 MiB fill)",
                       "parallelism": "external momenta sharded over GPUs (64 per GPU), no collective",
                       "integrals_per_step_per_gpu": n_out, "nominal_evals_per_step_per_gpu": evals},
            "integrals_per_s": whole_job_rate(world, n_out, ms),
            "clocks": clocks, "gpu_launches": 5 * args.steps,  # phi-rows pre-pass, psi pre-pass, the two moment kernels (one returns at once), fix-up
            "e2e": {"value": whole_job_rate(world, evals, e2e_s * 1e3), "unit": UNIT, "h2d_bytes_per_step": h2d,
                    "d2h_bytes_per_step": d2h, "ms_per_step": e2e_s * 1e3, "s1_host_ms": t_s1 * 1e3},
            "roofline": roof,
            "wall_s_timed_region": t_wall}

    if not args.no_others and world == 1:
        line["other_configs"] = time_other_configs(torch, B, inputs, make_rules, peak)

    parity_ok = True
    if (args.full or not args.no_cpu_baseline) and world == 1:
        # the oracle as it stands, on the host cores, on the SAME nodes the GPU used (R: the library's dfrg_quad_nodes)
        import oracle
        from oracle.harness import RTOL, SENS_EPS, oracle_run, parity_report
        per_out = evals // n_out
        if args.full:
            sel = np.arange(n_out, dtype=np.int64)
        else:
            probe_sel = np.arange(0, n_out, n_out // 256)[:256]
            t0 = time.perf_counter()
            oracle_run(c, R, sel=probe_sel)
            rate = probe_sel.size / (time.perf_counter() - t0)                 # outputs per second
            n_s = int(min(n_out // 4, max(256, rate * 15.0)))               # about 15 s of host time
            stride = n_out // n_s
            stride += 1 - stride % 2                                         # odd: the sample visits every field-point residue
            sel = np.arange(0, n_out, stride, dtype=np.int64)[:n_s]
        t0 = time.perf_counter()
        o = oracle_run(c, R, sel=sel)
        dt = time.perf_counter() - t0
        got = out.cpu().numpy().ravel()[sel]
        rep = parity_report(got, o["out"], o["dmin"], o["sens"])
        rep = {k_: v for k_, v in rep.items() if not k_.startswith("_")}
        parity_ok = (rep["n_nonfinite_gpu_only"] == 0 and rep["max_rel_regular"] <= RTOL and
                     rep["max_sens_ratio_regular"] <= SENS_EPS and rep["max_sens_ratio_singular"] <= SENS_EPS)
        line["cpu_baseline"] = {"value": sel.size * per_out / dt, "unit": UNIT, "cores": oracle.num_threads(),
                                "kind": "oracle", "seconds": dt,
                                "sample": ("all %d outputs" % n_out) if args.full else
                                          "%d of %d outputs (every %dth), %d nodes each" % (sel.size, n_out, stride, per_out),
                                "nodes": "the library's (dfrg_quad_nodes), the same arrays the GPU call used",
                                "max_rel_err_vs_gpu_regular": rep["max_rel_regular"],
                                "max_abs_err_over_sens": max(rep["max_sens_ratio_regular"], rep["max_sens_ratio_singular"]),
                                "n_regular": rep["n_regular"], "n_pole": rep["n_pole"], "n_cancelling": rep["n_cancelling"],
                                "max_rel_cancelling": rep["max_rel_cancelling"],
                                "max_abs_err_over_sens_singular": rep["max_sens_ratio_singular"],
                                "n_nonfinite_gpu_only": rep["n_nonfinite_gpu_only"],
                                "bars": {"rel_regular": RTOL, "abs_over_sens": SENS_EPS}, "parity_ok": parity_ok}
        if args.report:
            with open(args.report, "w") as fh:
                json.dump({"workload": WORKLOAD, "compared": int(sel.size), "of": n_out, "oracle_seconds": dt, **rep,
                           "bars": {"rel_regular": RTOL, "abs_over_sens": SENS_EPS}, "parity_ok": parity_ok}, fh, indent=1)
    print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()
    return 0 if parity_ok else 1


if __name__ == "__main__":
    sys.exit(main())
