#!/usr/bin/env python
"""Benchmark of the column-generation VMAT hot path (BASELINE.json: "CG iterations/s and plan wall-time;
pricing SpMV GB/s vs B200 HBM peak").

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config prostate] [--impl reference]

One STEP = one whole plan optimisation on the seeded synthetic phantom: every column-generation
iteration (price -> leaf search -> aperture column -> master) until each beam holds an aperture
(configs[1], prostate-like: 180 iterations).  `value` = column-generation iterations per second with
D resident in HBM; `e2e` = the same through the C ABI from pinned HOST buffers (vmat_create's upload
and re-layout, the solve, the read-back of the plan, vmat_destroy all inside the timed region).
N > 1 runs N independent replicas (the path does not shard; no collective).
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "column_generation_iterations_per_s"
UNIT = "iterations/s"


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


# A number cited from a committed capture, not measured by the run that prints it: `ncu --set full` of k_price_spmv on
# configs[1], dram__bytes_read.sum + dram__bytes_write.sum of the FIRST pricing launch of a plan (all 180 beams
# un-occupied; 994,678,664 algorithmic bytes).  The kernel and the layout of D have not changed since that capture.
NCU_TRAFFIC_BYTES_FIRST_LAUNCH = {"prostate": 992094976 + 4541440}
NCU_TRAFFIC_SOURCE = "profiles/r02_price_spmv.md (ncu --set full of k_price_spmv<16,4,128>, round 2)"


class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.proc = index, None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.proc = None

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            out, _ = self.proc.communicate(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
            out, _ = self.proc.communicate()
        sm, mx, reasons = [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for line in out.strip().splitlines():
            f = [x.strip() for x in line.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1]))
            except ValueError:
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(mx)), "reasons": sorted(reasons),
                "samples": len(sm)}


def pricing_algorithmic_bytes(nnz, B, V, N, iters):
    """at outer iteration t the product streams the rows of the N-t un-occupied beams:
    (N-t)/N * (8 nnz + 8 B + 4 B) + 4 V bytes (values + indices, row pointers, g out, one read of w)."""
    return [(N - t) / N * (8.0 * nnz + 12.0 * B) + 4.0 * V for t in range(iters)]


def make_inputs(config: str, seed: int = 0):
    import vmat_inputs

    t0 = time.perf_counter()
    ph = vmat_inputs.make_phantom(config, seed=seed)
    return ph, time.perf_counter() - t0


def oracle_sample(ph, budget_s: float, chunk: int = 5, threads: int = 0):
    """The oracle as it stands on the first iterations of the same workload, until `budget_s` of CPU work (the whole
    plan if the budget allows).  threads > 0: run it on that many OpenMP threads."""
    from oracle import Oracle, vmat_oracle

    all_threads = vmat_oracle.num_threads()
    if threads > 0:
        vmat_oracle.set_num_threads(threads)
    try:
        return _oracle_sample(ph, budget_s, chunk)
    finally:
        vmat_oracle.set_num_threads(all_threads)


def _oracle_sample(ph, budget_s: float, chunk: int):
    from oracle import Oracle, vmat_oracle

    o = Oracle.from_phantom(ph)
    plan = None
    done, t_used = 0, 0.0
    cost = float("nan")
    while done < ph.config.n_beams and t_used < budget_s:
        t0 = time.perf_counter()
        occ, l, r, y, z, tr = o.solve(chunk, plan=plan)
        t_used += time.perf_counter() - t0
        if tr.iters == 0:
            break
        done += tr.iters
        cost = float(tr.cost[-1])
        plan = (occ, l, r, y)
    return done, t_used, vmat_oracle.num_threads(), cost


def run_reference(args):
    """--impl reference: the CPU oracle on the host cores, same config / metric / unit (rank 0 only)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    ph, _ = make_inputs(args.config)
    budget = args.ref_budget_s
    for _ in range(args.warmup):
        oracle_sample(ph, min(2.0, budget))
    it_total, t_total, cores = 0, 0.0, 1
    for _ in range(args.steps):
        it, t, cores, _ = oracle_sample(ph, budget)
        it_total += it
        t_total += t
    value = it_total / t_total
    sample = (f"first {it_total // max(args.steps, 1)} of {ph.config.n_beams} column-generation iterations per step "
              f"(~{budget:.0f} s of CPU work), oracle/vmat_oracle.c as it stands (fp64, OpenMP)")
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * t_total / max(args.steps, 1),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": workload_config(ph, args),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


def aggregate_over_ranks(ms, done_iters, launches, dist, device):
    """Replicas: the job's time is the MAX over ranks of the device-timed region, its
    work the SUM of the iterations (and kernel launches) every rank completed.  No data-path collective."""
    if dist is None:
        return float(ms), int(done_iters), int(launches)
    import torch

    t = torch.tensor([ms], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    n = torch.tensor([done_iters, launches], device=device, dtype=torch.int64)
    dist.all_reduce(n)
    return float(t.item()), int(n[0].item()), int(n[1].item())


def run_sweep(args):
    """BASELINE.json configs[3]: the pricing product g = D w in isolation on synthetic beamlet-major CSR
    (row lengths U[200,800], voxel ids in runs of 8-64, w ~ N(0,1)), and the leaf-row search on 180 x 40 rows of
    40-80 beamlets.  One JSON line per point; GB/s = algorithmic bytes (8 nnz + 12 rows + 4 V) / kernel time."""
    import torch

    import __graft_entry__ as entry

    entry.build()
    import paper_1005_4396_b200 as vm
    import vmat_inputs

    torch.cuda.set_device(0)
    peak, peak_src = load_peaks()
    R, C = 80, 200                                     # rows are grouped as "beams" of R*C beamlets
    for nnz_target in [int(float(x)) for x in args.sweep_nnz.split(",")]:
        for V in [int(float(x)) for x in args.sweep_voxels.split(",")]:
            row_ptr, col, val = vmat_inputs.make_sweep_matrix(nnz_target, V, seed=0)
            rows = row_ptr.size - 1
            N = (rows + R * C - 1) // (R * C)
            row_ptr = np.concatenate([row_ptr, np.full(N * R * C - rows, row_ptr[-1], np.int64)])
            w = vmat_inputs.make_normal(V, seed=1)
            # alpha = beta = 1 and T = -w/2 make the empty plan's own penalty gradient (Eq. 1 at z = 0) equal w
            # exactly, so vmat_price_spmv(NULL) is the kernel alone (no staging of a caller-supplied gradient)
            one = np.ones(V, np.float32)
            opt = vm.default_options()
            opt.validate = 0
            plan = vm.Plan.create(row_ptr, col, val, (-0.5 * w).astype(np.float32), one, one,
                                  np.arange(N, dtype=np.float64), R, C, 2, 0.1, options=opt)
            g = torch.empty(N * R * C, dtype=torch.float32, device="cuda")
            wd = torch.empty(V, dtype=torch.float32, device="cuda")
            plan.dose(None, wd)
            assert np.array_equal(wd.cpu().numpy(), w), "plan gradient differs from the sweep's w"
            for _ in range(3):
                plan.price_spmv(g)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            nrep = 10
            e0.record()
            for _ in range(nrep):
                plan.price_spmv(g)
            e1.record()
            torch.cuda.synchronize()
            us = e0.elapsed_time(e1) * 1e3 / nrep
            nnz = int(row_ptr[-1])
            alg = 8.0 * nnz + 12.0 * rows + 4.0 * V
            # spot check against the definition on a few rows (fp64 on the host, not the oracle: a plain dot)
            gh = g.cpu().numpy()
            for i in np.random.default_rng(0).integers(0, rows, 50):
                a, b = row_ptr[i], row_ptr[i + 1]
                ref = float(np.dot(val[a:b].astype(np.float64), w[col[a:b]].astype(np.float64)))
                mag = float(np.dot(np.abs(val[a:b]).astype(np.float64), np.abs(w[col[a:b]]).astype(np.float64)))
                assert abs(gh[i] - ref) <= 1e-5 * mag + 1e-30, (i, gh[i], ref)
            print(json.dumps({"sweep": "pricing_spmv", "nnz": nnz, "rows": rows, "voxels": V, "us": us,
                              "GBs": alg / us / 1e3, "frac_of_peak": alg / us / 1e3 / peak, "peak": peak,
                              "peak_source": peak_src, "algorithmic_bytes": alg,
                              "support_voxels": plan.n_support}), flush=True)
            plan.destroy()
            del g, wd
            torch.cuda.empty_cache()
    # leaf-row search on 180 x 40 rows
    for Cs in (40, 60, 80):
        N, Rs = 180, 40
        B = N * Rs * Cs
        opt = vm.default_options()
        plan = vm.Plan.create(np.zeros(B + 1, np.int64), np.zeros(1, np.int32), np.zeros(1, np.float32),
                              np.zeros(4, np.float32), np.zeros(4, np.float32), np.zeros(4, np.float32),
                              np.arange(N, dtype=np.float64) * 2.0, Rs, Cs, 2, 0.1, options=opt)
        gd = torch.from_numpy(vmat_inputs.make_search_rows(N, Rs, Cs, seed=0)).cuda()
        al = torch.zeros(N * Rs, dtype=torch.int32, device="cuda")
        ar = torch.zeros(N * Rs, dtype=torch.int32, device="cuda")
        bp = torch.zeros(N, dtype=torch.float64, device="cuda")
        for _ in range(3):
            plan.leaf_search(gd, al, ar, bp)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        nrep = 50
        e0.record()
        for _ in range(nrep):
            plan.leaf_search(gd, al, ar, bp)
        e1.record()
        torch.cuda.synchronize()
        us = e0.elapsed_time(e1) * 1e3 / nrep
        print(json.dumps({"sweep": "leaf_search", "beams": N, "leaf_rows": Rs, "leaf_cols": Cs, "us": us,
                          "rows_per_s": N * Rs / (us * 1e-6)}), flush=True)
        plan.destroy()


def workload_config(ph, args):
    c = ph.config
    return {
        "workload": f"configs[{ {'tiny': 0, 'prostate': 1, 'hn': 2, 'stress': 4}[c.name] }] {c.name}-like phantom, "
                    f"{c.n_beams} column-generation iterations per step",
        "grid": list(c.grid), "voxel_mm": c.voxel_mm, "beams": c.n_beams, "leaf_rows": c.n_rows, "leaf_cols": c.n_cols,
        "beamlets": ph.n_beamlets, "voxels": ph.n_voxels, "nnz": ph.nnz, "max_leaf_travel": c.max_leaf_travel,
        "gamma": c.gamma, "seed": ph.seed,
        "l2": "inputs larger than L2 (D streams >= 0.5 GB per iteration on average); no flush",
        "parallelism": "replicas" if args.gpus > 1 else "single GPU",
    }


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default="prostate", choices=["tiny", "prostate", "hn", "stress"])
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--cpu-budget-s", type=float, default=150.0,
                    help="cap on the CPU seconds of the cpu_baseline leg (the oracle's whole plan if it fits)")
    ap.add_argument("--cpu-single-thread-s", type=float, default=10.0,
                    help="CPU seconds of the single-thread prefix of the cpu_baseline leg (0: skip)")
    ap.add_argument("--ref-budget-s", type=float, default=15.0, help="CPU seconds per step of --impl reference")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--master-mode", type=int, default=None, choices=[0, 1],
                    help="vmat_options.master_mode: 0 conjugate directions, 1 Newton on the reduced problem (the library's default)")
    ap.add_argument("--d-format", type=int, default=None, choices=[0, 1],
                    help="vmat_options.d_format: 0 fp32 CSR (the headline layout), 1 aligned slot pairs with 16-bit ids")
    ap.add_argument("--sweep", action="store_true", help="configs[3]: isolated pricing / search kernel sweep")
    ap.add_argument("--sweep-nnz", default="5e7,1e8,2.5e8,5e8,1e9")
    ap.add_argument("--sweep-voxels", default="1048576,2097152,4194304")
    args = ap.parse_args()
    if args.sweep:
        return run_sweep(args)
    if args.warmup < 3 and args.impl == "b200":
        args.warmup = 3
    if args.impl == "reference":
        return run_reference(args)

    import torch

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the hot path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist

        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    import __graft_entry__ as entry

    entry.build()
    import paper_1005_4396_b200 as vm

    ph, gen_s = make_inputs(args.config)
    c = ph.config
    iters = c.n_beams                      # S5: one aperture per beam
    # pinned host copies of the problem (the e2e leg uploads from these every step)
    host = [torch.from_numpy(a).pin_memory() for a in (ph.row_ptr, ph.col_idx, ph.val, ph.T, ph.alpha, ph.beta)]
    h2d_bytes = int(sum(t.numel() * t.element_size() for t in host) + ph.theta_deg.nbytes)
    d2h_bytes = int(c.n_beams * (1 + 8 + 2 * 4 * c.n_rows) + 3 * 8)

    def create(record_phases=0):
        opt = vm.default_options()
        opt.record_phases = record_phases
        if args.master_mode is not None:
            opt.master_mode = args.master_mode
        if args.d_format is not None:
            opt.d_format = args.d_format
        return vm.Plan.create(*[t.numpy() for t in host], ph.theta_deg, c.n_rows, c.n_cols, c.max_leaf_travel, c.gamma,
                              options=opt)

    empty = (np.zeros(c.n_beams, np.uint8), np.zeros((c.n_beams, c.n_rows), np.int32),
             np.zeros((c.n_beams, c.n_rows), np.int32), np.zeros(c.n_beams))

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident leg: `value` -----------------------------------------------------------
    t0 = time.perf_counter()
    plan = create()
    torch.cuda.synchronize()
    create_ms = 1e3 * (time.perf_counter() - t0)
    stream = torch.cuda.current_stream()
    last = None
    for _ in range(args.warmup):
        plan.set_plan(*empty)
        last = plan.solve(iters, trace=False)
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
    barrier()
    l0 = plan.launch_count
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record(stream)
    done_iters = 0
    for _ in range(args.steps):
        plan.set_plan(*empty)
        last = plan.solve(iters, trace=False)
        done_iters += last.iters
    ev1.record(stream)
    barrier()
    ms = ev0.elapsed_time(ev1)
    launches = plan.launch_count - l0
    ms, done_iters, launches = aggregate_over_ranks(ms, done_iters, launches, dist, "cuda")
    clocks = sampler.stop() if rank == 0 else None
    value = done_iters / (ms * 1e-3)
    final_cost = last.cost

    # ---- per-phase device times (CUDA events on the plan's stream) and the pricing roofline -------
    plan.destroy()
    plan = create(record_phases=1)
    plan.set_plan(*empty)
    plan.solve(iters, trace=False)
    ph_us = {"price": 0.0, "search": 0.0, "column": 0.0, "master": 0.0, "total": 0.0}
    inner_total = 0
    m_passes = m_bytes = m_cg = 0.0
    m_clk = [0.0, 0.0, 0.0]
    for _ in range(args.steps):
        plan.set_plan(*empty)
        st = plan.solve(iters, trace=True)
        for k, v in (("price", st.us_price), ("search", st.us_search), ("column", st.us_column),
                     ("master", st.us_master), ("total", st.us_total)):
            ph_us[k] += v / args.steps
        inner_total += int(st.inner.sum())
        m_passes += st.master_passes / args.steps
        m_bytes += st.master_bytes / args.steps
        m_cg += st.master_cg_steps / args.steps
        for i, v in enumerate((st.master_clk_cg, st.master_clk_wait, st.master_clk_load)):
            m_clk[i] += v / args.steps
    # ---- steps (a)+(b) on the finished plan, both layouts (north_star: "chosen by measurement") -------------
    occ_f, left_f, right_f, _ = plan.get_plan()
    nnz_open = 0
    for k in range(c.n_beams):
        for r in range(c.n_rows):
            i0 = (k * c.n_rows + r) * c.n_cols
            nnz_open += int(ph.row_ptr[i0 + right_f[k, r]] - ph.row_ptr[i0 + left_f[k, r]])
    dose = {"nnz_exposed": nnz_open, "exposed_fraction_of_nnz": nnz_open / ph.nnz}
    for name, path in (("columns", 0), ("direct_atomics", 1)):
        for _ in range(3):
            plan.dose_recompute(path)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        nrep = 20
        e0.record(stream)
        for _ in range(nrep):
            plan.dose_recompute(path)
        e1.record(stream)
        torch.cuda.synchronize()
        dose[name + "_us"] = e0.elapsed_time(e1) * 1e3 / nrep
    # algorithmic bytes of the direct pass: the exposed rows (8 B per entry) + z, w out and T, alpha, beta in
    dose_bytes = 8.0 * nnz_open + 20.0 * plan.n_support
    dose["direct_atomics_GBs"] = dose_bytes / dose["direct_atomics_us"] / 1e3
    dose["direct_algorithmic_bytes"] = dose_bytes
    plan.dose_recompute(0)
    alg = pricing_algorithmic_bytes(ph.nnz, ph.n_beamlets, ph.n_voxels, c.n_beams, iters)
    peak, peak_src = load_peaks()
    achieved = sum(alg) / (ph_us["price"] * 1e-6) / 1e9
    roofline = {
        "kernel": "k_price_spmv<16,4> (pricing SpMV, step c)",
        "bound": "hbm", "achieved": achieved, "peak": peak,
        "unit": "GB/s", "frac": achieved / peak, "frac_of_8TBs_nominal": achieved / 8000.0,
        "traffic": NCU_TRAFFIC_BYTES_FIRST_LAUNCH.get(c.name),
        "traffic_source": NCU_TRAFFIC_SOURCE if c.name in NCU_TRAFFIC_BYTES_FIRST_LAUNCH else None,
        "traffic_note": "cited from that capture, not measured by this run: ncu dram bytes of the FIRST launch of a "
                        "plan (compare algorithmic_bytes_first_launch)",
        "peak_source": peak_src,
        "algorithmic_bytes_per_launch_avg": sum(alg) / iters, "algorithmic_bytes_first_launch": alg[0],
        "avg_launch_us": ph_us["price"] / iters, "launches_per_step": iters,
        "how": "CUDA events on the plan's stream around every pricing launch of the phase-timed steps",
    }
    # the master kernel (step e) takes the larger share of a plan: its algorithmic traffic = the touched 512-byte
    # segments of the aperture-dose columns x the passes that multiplied them (counted on the device); on
    # configs[1] those segments sit in shared memory, so this is an effective rate, not DRAM traffic
    m_gbs = m_bytes / (ph_us["master"] * 1e-6) / 1e9 if ph_us["master"] > 0 else 0.0
    newton = m_cg > 0
    roofline_master = {
        "kernel": ("k_newton" if newton else "k_master") + " (master solve, steps a+b+e)", "bound": "hbm",
        "achieved": m_gbs, "peak": peak, "unit": "GB/s",
        "frac": m_gbs / peak, "traffic": None, "algorithmic_bytes_per_step": m_bytes, "passes_per_step": m_passes,
        "us_per_pass": ph_us["master"] / m_passes if m_passes else None, "launches_per_step": iters,
        "note": ("latency bound: a solve is two or three passes over the touched column segments, each followed by "
                 "conjugate-gradient steps on the K x K reduced problem in one block (DESIGN.md section 7); "
                 if newton else
                 "latency bound: two grid barriers and two control steps per inner iteration; ") +
                "bytes = touched column segments x passes, device-counted",
    }
    if newton:
        clk_us = (clocks or {}).get("sm_mhz") or 1965.0
        roofline_master.update({"cg_steps_per_step": m_cg, "cg_us_per_step": m_clk[0] / clk_us,
                                "waiting_for_passes_us_per_step": m_clk[1] / clk_us,
                                "loading_hessian_us_per_step": m_clk[2] / clk_us})
    phases = {k + "_us_per_step": v for k, v in ph_us.items()}
    phases["master_inner_iterations_per_step"] = inner_total / args.steps
    info = {"nnz": plan.nnz, "nnz_padded": plan.nnz_padded, "support_voxels": plan.n_support,
            "device_bytes": plan.device_bytes, "d_format": int(args.d_format or 0), "pricing_bytes": plan.pricing_bytes,
            "pricing_bytes_per_entry": plan.pricing_bytes / max(plan.nnz, 1)}
    plan.destroy()

    # ---- end-to-end leg from pinned host buffers ----------------------------------------------------
    e2e = None
    if not args.no_e2e:
        def e2e_step():
            p = create()
            s = p.solve(iters, trace=False)
            out = p.get_plan()
            p.destroy()
            return s, out

        e2e_step()
        barrier()
        t0 = time.perf_counter()
        n_e2e = max(1, min(args.steps, 3))
        it_e2e = 0
        for _ in range(n_e2e):
            s, _ = e2e_step()
            it_e2e += s.iters
        barrier()
        dt = time.perf_counter() - t0
        dt, it_e2e, _ = aggregate_over_ranks(dt, it_e2e, 0, dist, "cuda")
        e2e = {"value": it_e2e / dt, "unit": UNIT, "h2d_bytes_per_step": h2d_bytes, "d2h_bytes_per_step": d2h_bytes,
               "ms_per_step": 1e3 * dt / n_e2e, "steps": n_e2e,
               "what": "vmat_create from pinned host CSR + vmat_solve + vmat_get_plan + vmat_destroy, wall clock"}

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    cpu_baseline = None
    if not args.no_cpu_baseline and world == 1:
        it, t, cores, ocost = oracle_sample(ph, args.cpu_budget_s)
        whole = it >= c.n_beams
        cpu_baseline = {"value": it / t, "unit": UNIT, "cores": cores, "kind": "oracle", "nproc": os.cpu_count(),
                        "sample": (f"the whole plan, {it} column-generation iterations" if whole else
                                   f"first {it} of {c.n_beams} column-generation iterations") +
                                  f" of the same phantom ({t:.1f} s), oracle/vmat_oracle.c as it stands (fp64, OpenMP)",
                        "iterations": it, "seconds": t, "whole_plan": whole, "final_cost": ocost}
        if args.cpu_single_thread_s > 0:
            it1, t1, _, _ = oracle_sample(ph, args.cpu_single_thread_s, chunk=2, threads=1)
            cpu_baseline["single_thread"] = {"value": it1 / t1, "unit": UNIT, "cores": 1,
                                             "sample": f"first {it1} iterations on one thread ({t1:.1f} s)"}

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic", "config": workload_config(ph, args),
        "plan_wall_time_ms": ms / args.steps, "final_cost": final_cost,
        "roofline": roofline, "cpu_baseline": cpu_baseline, "e2e": e2e, "gpu_launches": launches, "clocks": clocks,
        "roofline_master": roofline_master, "phases": phases, "dose_pass": dose, "layout": info, "create_ms": create_ms, "generate_inputs_s": gen_s,
        "paper_context": "PAPER.md:157 whole plan 18-31 s (CUDA, Tesla C1060) / 5-8 min (MATLAB, Xeon) on clinical "
                         "cases of 1.8e7-5.5e7 non-zeros; different machine and data, not a target",
    }
    print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
