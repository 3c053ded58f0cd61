#!/usr/bin/env python
"""bench.py -- one JSON line for the hot path of arXiv 2304.06340 on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 2] [--impl reference]

A *step* is one pass of the whole hot path (every row of SURVEY.md 8(a)) on BASELINE.json's config 2 (the
configuration the metric is quoted on; icosphere level 4, 6-pt rule, 30,720 sources, 128x64x128 = 1,048,576 ball
quadrature nodes on [0,128]):

    sfd_mesh_icosphere(level)                               A1/A2
    for s in config.s:  sfd_weak_distance(eps = 0)          A3 + frequency nodes + A4 direct sum + A6
    for s in config.s:  sfd_weak_distance(eps = 1e-9)       A3 + frequency nodes + A5 type-3 NUFFT + A6

`value` = source.frequency pairs per second = the pairs the step actually COMPUTES (the direct-sum evaluations: J * K_eval
each, K_eval = the nodes the library visits, sfd_weak_distance_targets: the xi_3 >= 0 half of the rule, mirror nodes give
equal terms) / the whole step's device time.  The NUFFT evaluations compute no pairs: they are reported as ms per
distance and as `equivalent_pairs_per_s` (J * K_eval / their time), labelled as such, and do not enter `value`.
`e2e` = the same through the host-buffer C-ABI calls (sfd_weak_distance_host: mesh copied from pinned host memory,
distance copied back, inside the timed region).  `roofline` describes the dominant kernel (direct_sum_kernel, FP64-ALU
bound); `roofline_nufft` lists the HBM-judged type-3 stages.  `cpu_baseline` times the oracle (oracle/, as it stands) on
a bounded sample of the same nodes on this box's host cores.

The default invocation then also times, once per tolerance, BASELINE.json's config 3 -- the "full level-6 distance
evaluation in ms" of the north star -- and config 5 at level 8 (`ms_per_distance`, `stage_ms`, `roofline_nufft`).
`ms_per_distance` is the library's default mode (the target sort of a type-3 evaluation runs beside the spreader and the
FFT passes on a second stream); `stage_ms` and the NUFFT rooflines come from a pass with every stage on one stream.
`--config 5` emits one JSON line per level 0..8 and s (distance, h, ms) before the summary line.

Multi-GPU (torchrun, --gpus N): the frequency nodes of every distance are sharded over the ranks by radial shell
(sharding.weak_distance_sharded -> sfd_weak_distance_range per rank, one all-reduce of a 16-byte device pair): strong
scaling of the same step.  `--replicas` times N independent copies instead (weak scaling, no collective).
`--simulate-ranks N` (one GPU) evaluates the N shards one after the other and reports each shard's device time.
"""
import argparse
import ctypes as C
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

import workloads  # noqa: E402

METRIC = "source*frequency pairs/s (fp64 nuhat)"
UNIT = "pairs/s"
PROBE_SRC = os.path.join(ROOT, "bench_probe.cu")
PROBE_LIB = os.path.join(ROOT, "libbench_probe.so")


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=2, help="BASELINE.json config number (2 = the headline)")
    ap.add_argument("--impl", default="sfd", choices=["sfd", "reference"])
    ap.add_argument("--workload", default="config", choices=["config", "fig4a", "fig4b", "exact_a", "exact_b"],
                    help="config: BASELINE.json config (default); fig4a / fig4b: the paper's own timing experiments "
                         "(P:244: N = 7, M = 128 / N = 5, M = 416; xi_max = 5, 64-pt rule, eps 1e-7); exact_a / exact_b: "
                         "the exact-formula direct summation the paper quotes from [38] (P:244: ~100,000 triangles, "
                         "M = 100 / 80 triangles, M = 400)")
    ap.add_argument("--precision", default="fp64", choices=["fp64", "fp32"],
                    help="arithmetic of the NUFFT grids (fig4a / fig4b only; the paper ran its NUFFT in fp32, P:238)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-extras", action="store_true", help="skip the config-3 / config-5 distances of the default run")
    ap.add_argument("--cpu-seconds", type=float, default=12.0, help="target CPU time of the oracle sample")
    ap.add_argument("--replicas", action="store_true",
                    help="multi-GPU: N independent evaluations (weak scaling, no collective) instead of the sharded path")
    ap.add_argument("--force-sharded", action="store_true",
                    help="run the sharded code path (sfd_weak_distance_range + combine) even with one rank: a self-test")
    ap.add_argument("--simulate-ranks", type=int, default=0,
                    help="one GPU: evaluate the shards of an N-rank run one after the other and report their device times")
    return ap.parse_args()


def workload(cfg_id, level=None):
    c = workloads.CONFIGS[cfg_id]
    if level is None:
        level = c["level"] if isinstance(c["level"], int) else max(c["level"])
    F = 20 * 4 ** level
    J = F * c["rule"]
    K = c["n_r"] * c["n_theta"] * c["n_phi"]
    return c, level, J, K


def k_evaluated(c):
    """Nodes a distance evaluation visits (include/sfd.h sfd_weak_distance_targets): the xi_3 >= 0 half, even n_phi."""
    if c["n_phi"] % 2:
        return c["n_r"] * c["n_theta"] * c["n_phi"]
    return c["n_r"] * (c["n_theta"] - c["n_theta"] // 2) * c["n_phi"]


def config_dict(cfg_id, n_gpus, mode="single"):
    """The same dictionary for both arms (sfd and reference): the workload, and how it is spread over GPUs."""
    c, level, J, K = workload(cfg_id)
    par = {"single": "1 GPU",
           "sharded": f"frequency nodes sharded over {n_gpus} ranks by radial shell, 1 all-reduce of 16 B per distance",
           "replicas": f"{n_gpus} independent distance evaluations (one per GPU), no collective"}[mode]
    return {"workload": f"BASELINE.json config {cfg_id}: icosphere level {level}, {c['rule']}-pt rule, J={J} sources; "
                        f"ball quadrature {c['n_r']}x{c['n_theta']}x{c['n_phi']} on [0,{c['R']:g}], K={K} nodes",
            "level": level, "rule": c["rule"], "J": J, "K": K, "R": c["R"],
            "n_r": c["n_r"], "n_theta": c["n_theta"], "n_phi": c["n_phi"], "s": list(c["s"]), "eps": list(c["eps"]),
            "K_evaluated": k_evaluated(c),
            "symmetry": "nodes with xi_3 >= 0 only, doubled weights (mirror nodes give equal terms; DESIGN.md R18)",
            "parallelism": par,
            "l2": "L2 flushed (512 MiB memset) between timed steps; NUFFT grids (0.75 GB) also exceed L2"}


# ---------------------------------------------------------------------------------------------------------------
# bench-side helper: the FP64 FMA peak of the device (not part of libsfd.so)
def build_probe(force=False):
    if force or not os.path.exists(PROBE_LIB) or os.path.getmtime(PROBE_LIB) < os.path.getmtime(PROBE_SRC):
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        subprocess.run([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-shared", "-Xcompiler",
                        "-fPIC", PROBE_SRC, "-o", PROBE_LIB], check=True)
    return PROBE_LIB


def probe_fp64(stream_ptr, iters=8192):
    lib = C.CDLL(build_probe())
    lib.bench_probe_fp64.restype = C.c_int
    lib.bench_probe_fp64.argtypes = [C.c_int, C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_double)]
    tf, ms = C.c_double(), C.c_double()
    rc = lib.bench_probe_fp64(iters, C.c_void_p(stream_ptr), C.byref(tf), C.byref(ms))
    if rc != 0:
        raise RuntimeError(f"bench_probe_fp64 failed ({rc})")
    return tf.value, ms.value


def measured_traffic(kernel, wl):
    """dram read + write bytes per launch of `kernel` on workload `wl`, from the committed ncu --set full summary
    profiles/traffic.csv (kernel,workload,dram_bytes_read,dram_bytes_write,source); None when no capture is recorded."""
    try:
        with open(os.path.join(ROOT, "profiles", "traffic.csv")) as f:
            for line in f:
                p = [t.strip() for t in line.split(",")]
                if len(p) >= 4 and p[0] == kernel and p[1] == wl:
                    return int(float(p[2])) + int(float(p[3]))
    except OSError:
        pass
    return None


# ---------------------------------------------------------------------------------------------------------------
# reference arm / cpu_baseline: the oracle, as it stands, on a bounded sample of the workload
def oracle_sample(cfg_id, seconds, steps=1, warmup=0):
    """Times oracle.direct_sum (+ mesh, nodes, reduce) on K_sub seeded nodes x all J sources.  The nodes are drawn from the
    ones the GPU arm evaluates (the xi_3 >= 0 half of the rule).  Returns (pairs_per_s, ms_per_step, cores, sample, K_sub)."""
    sys.path.insert(0, os.path.join(ROOT, "oracle"))
    import sfd_oracle as O
    c, level, J, K = workload(cfg_id)
    V, F = O.mesh_icosphere(level)
    if c["jitter"]:
        V = workloads.jitter_vertices(V, F, *c["jitter"])
    x, w = O.nodes(V, F, c["rule"])
    xi, W = O.freq_nodes(c["n_r"], c["n_theta"], c["n_phi"], c["R"])
    if c["n_phi"] % 2 == 0:   # the half the library visits: rings b >= n_theta // 2 (mu ascending), weights doubled
        g = np.arange(K).reshape(c["n_r"], c["n_theta"], c["n_phi"])[:, c["n_theta"] // 2:, :].reshape(-1)
        xi, W = np.ascontiguousarray(xi[g]), np.ascontiguousarray(2.0 * W[g])
    Kh = len(W)
    cores = O.num_threads()
    # calibrate on 64 nodes, then size the sample for ~`seconds` of CPU work
    idx = workloads.target_subset(Kh, 64, seed=1)
    t0 = time.perf_counter()
    O.direct_sum(x, w, xi[idx])
    rate = 64 * J / (time.perf_counter() - t0)
    k_sub = int(min(Kh, max(64, seconds * rate / J)))
    idx = workloads.target_subset(Kh, k_sub, seed=0)
    xs, Ws = np.ascontiguousarray(xi[idx]), np.ascontiguousarray(W[idx])
    times = []
    for it in range(warmup + steps):
        t0 = time.perf_counter()
        Vs, Fs = O.mesh_icosphere(level)
        xo, wo = O.nodes(Vs if not c["jitter"] else V, Fs, c["rule"])
        nu = O.direct_sum(xo, wo, xs)
        for s in c["s"]:
            O.reduce(nu, xs, Ws, s)
        dt = time.perf_counter() - t0
        if it >= warmup:
            times.append(dt)
    t = float(np.mean(times))
    sample = (f"oracle mesh+nodes+direct_sum+reduce on {k_sub} of the {Kh} evaluated nodes (SplitMix64 seed 0) x all {J} "
              f"sources, {k_sub * J:.3e} pairs per step")
    return k_sub * J / t, t * 1e3, cores, sample, k_sub


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    per_step = max(2.0, min(20.0, 120.0 / max(1, args.steps + args.warmup)))
    v, ms, cores, sample, _ = oracle_sample(args.config, per_step, steps=args.steps, warmup=args.warmup)
    mode = "single" if args.gpus == 1 else ("replicas" if args.replicas else "sharded")
    line = {"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True,
            "scaling": "weak" if mode != "sharded" else "strong", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic", "config": config_dict(args.config, args.gpus, mode),
            "cpu_baseline": {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


# ---------------------------------------------------------------------------------------------------------------
class ClockSampler:
    """nvidia-smi clocks / throttle reasons of one GPU, sampled every 100 ms while the timed region runs."""
    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows, self.proc = [], None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(index), f"--query-gpu={self.FIELDS}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.perf_counter(), [f.strip() for f in line.split(",")]))

    def stop(self, t0, t1):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        rows = [r for (t, r) in self.rows if t0 <= t <= t1 and len(r) >= 7] or [r for (_, r) in self.rows if len(r) >= 7]
        if not rows:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        sm = sorted(float(r[0]) for r in rows)
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for i, n in enumerate(names) if any(r[3 + i].lower().startswith("active") for r in rows)]
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": float(rows[0][1]), "samples": len(rows),
                "power_w_max": max(float(r[2]) for r in rows), "reasons": reasons}


# FP64-pipe instructions per source.target pair of direct_sum_kernel (checked against the SASS of
# the inner loop).  sfd_weak_distance runs the ball-rule variant of that kernel (one direction and BALL_T = 16 radii per
# thread share the dot product dhat . x: direct.cu BALL).  Per pair: rounding addition and residual with the product r g
# inside them 2 DFMA + 1 DADD; f^2 1 DMUL; monic sin / cos polynomials 2 DADD + 2 DFMA + 1 DMUL; leading coefficients and
# weight 2 DMUL; rotation by the table entry and accumulation 4 DFMA.  Per source (/16): dot product 1 DMUL + 2 DFMA,
# weight x leading coefficients 2 DMUL  ->  (8 + 2/16) DFMA + (4 + 3/16) DMUL + 3 DADD = 15.31 FP64 instructions, 23.44 flops
# per pair.  The counts below are what the timed kernel executes.
BALL_T = 16
DFMA_PER_PAIR, DMUL_DADD_PER_PAIR = 8 + 2 / BALL_T, 7 + 3 / BALL_T
FLOPS_PER_PAIR = 2 * DFMA_PER_PAIR + DMUL_DADD_PER_PAIR
FP64_LANES_PER_SM = 64          # DFMA / clk / SM on B200 (nominal 37-40 TFLOP/s at 1.965 GHz x 148 SMs)


def nufft_rooflines(P, c, J, K, eps, st, ext, hbm_peak, hbm_src, sm_mhz, n_sms, tag):
    """Roofline entries of one type-3 evaluation: spread / FFT / interp against measured HBM with ALGORITHMIC bytes (DESIGN.md
    section 6), interp also against the shared-memory roof that binds it; then the one-pass HBM-bound stages."""
    out = []
    w, nf, n2 = P.sfd_surface_ft_plan(J, K, [ext] * 3, [c["R"]] * 3, eps)
    cell = 8      # ball-centred targets: real strengths, real fine grid
    fine = nf[0] * nf[1] * nf[2] * cell
    no = [min(n2[d], n2[d] // 2 + w + 3 + (w & 1)) for d in range(3)]
    no[2] = no[2] - (n2[2] // 2 - (n2[2] // 4 - (w + 1) // 2 - 1))   # real strengths: only the upper z half is stored
    band = no[0] * no[1] * no[2]
    pa, pb = nf[0] * nf[1] * no[2], nf[0] * no[1] * no[2]
    sp_bytes = 2 * fine + 40 * J            # zero-fill + one accumulation pass of the grid + sorted sources
    ip_bytes = 16 * band + (32 + 16) * K    # the band of the inner grid, target records in, G out
    ft_bytes = fine + 16 * (2 * pa + 2 * pb + band)   # three passes: read non-zero rows, write the band
    smem_peak = 128.0 * n_sms * sm_mhz * 1e6 * 1e-9     # GB/s of shared memory, 128 B/clk/SM
    for name, kern, nbytes in (("spread", "spread_kernel", sp_bytes), ("fft", "fft_pass_kernel x3", ft_bytes),
                               ("interp", "interp_kernel", ip_bytes)):
        if name not in st or st[name] <= 0:
            continue
        ach = nbytes / (st[name] * 1e-3) * 1e-9
        e = {"kernel": kern, "workload": tag, "eps": eps, "w": w, "nf": nf[0], "n2": n2[0], "bound": "hbm",
             "achieved": ach, "peak": hbm_peak, "unit": "GB/s", "frac": ach / hbm_peak,
             "ms_per_launch": st[name], "algorithmic_bytes": nbytes, "peak_source": hbm_src}
        if name == "interp":   # the roof that actually binds the gather: 16 w^3 B of shared memory per target
            sm_ach = 16.0 * w ** 3 * K / (st[name] * 1e-3) * 1e-9
            e.update({"binding_roof": "shared memory", "smem_achieved_gbs": sm_ach, "smem_peak_gbs": smem_peak,
                      "smem_frac": sm_ach / smem_peak})
        out.append(e)
    # the one-pass HBM-bound stages around the transform (A3, frequency nodes, A5-9, A6), algorithmic bytes per unit
    for name, kern, nbytes in (("nodes", "nodes_kernel", 32 * J + 12 * (J // c["rule"])),
                               ("freq_nodes", "freq_expand_kernel", 32 * K),
                               ("post", "post_deconv_kernel", (24 + 32) * K),
                               ("reduce", "reduce_terms_kernel", 48 * K)):
        if name in st and st[name] > 0:
            ach = nbytes / (st[name] * 1e-3) * 1e-9
            out.append({"kernel": kern, "workload": tag, "eps": eps, "bound": "hbm", "achieved": ach, "peak": hbm_peak,
                        "unit": "GB/s", "frac": ach / hbm_peak, "ms_per_launch": st[name],
                        "algorithmic_bytes": nbytes, "peak_source": hbm_src})
    return out


def serial_stage_times(P, call, reps):
    """Stage times of a type-3 evaluation with every stage on the caller's stream (SFD_NO_OVERLAP=1: the library reads the
    variable at each call).  In the default mode, which is the one that is timed, the target sort runs beside the spreader
    and the FFT passes on a second stream, so those stages' event times contain it: the stages are attributed (and the
    NUFFT rooflines computed) from this serial pass, `ms_per_distance` from the default mode."""
    stages = {}
    os.environ["SFD_NO_OVERLAP"] = "1"
    try:
        for _ in range(reps):
            call()
            for name, t in P.sfd_last_stage_times():
                stages.setdefault(name, []).append(t)
    finally:
        os.environ.pop("SFD_NO_OVERLAP", None)
    return stages


def time_distances(P, torch, cfg_id, level, eps_list, s_list, reps, dist_fn=None, warm=1):
    """ms per distance (CUDA events on the launching stream), stage times and values of sfd_weak_distance on one config."""
    c, level, J, K = workload(cfg_id, level)
    q = (c["n_r"], c["n_theta"], c["n_phi"])
    V, F = P.sfd_mesh_icosphere(level)
    ext = 1.0
    if c["jitter"]:
        V = torch.as_tensor(workloads.jitter_vertices(V.cpu().numpy(), F.cpu().numpy(), *c["jitter"]), device=V.device)
        ext = 1.01
    wb = max(P.sfd_weak_distance_workspace(F.shape[0], c["rule"], q, c["R"], e, ext) for e in eps_list)
    work = torch.empty(wb, dtype=torch.uint8, device=V.device)
    out = {}
    fn = dist_fn or (lambda V, F, rule, s, R, q, eps, work: P.sfd_weak_distance(V, F, rule, s, R, q, eps, work=work))
    for eps in eps_list:
        for s in s_list:
            for _ in range(warm):
                fn(V, F, c["rule"], s, c["R"], q, eps, work)
            ms, stages = [], {}
            P.sfd_set_profiling(True)
            for _ in range(reps):
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record()
                d, I = fn(V, F, c["rule"], s, c["R"], q, eps, work)
                e1.record()
                torch.cuda.synchronize()
                ms.append(e0.elapsed_time(e1))
                for name, t in P.sfd_last_stage_times():
                    stages.setdefault(name, []).append(t)
            if eps > 0:
                stages = serial_stage_times(P, lambda: fn(V, F, c["rule"], s, c["R"], q, eps, work), reps)
            P.sfd_set_profiling(False)
            out[(eps, s)] = {"ms": float(np.median(ms)), "ms_best": float(min(ms)), "distance": d, "I": I,
                             "stage_ms": {k: float(np.median(v)) for k, v in stages.items()}}
    del work
    torch.cuda.empty_cache()
    return out, ext, J, K


def run_sfd(args):
    import torch
    import torch.distributed as dist
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the sfd arm has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    import paper_2304_06340_b200 as P
    from paper_2304_06340_b200 import sharding

    c, level, J, K = workload(args.config)
    q = (c["n_r"], c["n_theta"], c["n_phi"])
    R, rule = c["R"], c["rule"]
    eps_list = [e for e in c["eps"]]
    if args.config == 2:
        eps_list = [0.0, 1e-9]
    sharded = (world > 1 and not args.replicas) or args.force_sharded
    dev = torch.device("cuda", local)
    stream = torch.cuda.current_stream()

    # device-resident buffers, sized once (allocation is outside the timed region, like the paper's P:238)
    nV, nF, mesh_wb = P.sfd_mesh_icosphere_sizes(level)
    V = torch.empty((nV, 3), dtype=torch.float64, device=dev)
    F = torch.empty((nF, 3), dtype=torch.int32, device=dev)
    mesh_work = torch.empty(max(mesh_wb, 256), dtype=torch.uint8, device=dev)
    ext = 1.0 + (0.0 if not c["jitter"] else 0.01)
    if sharded:
        wb = 0
        for e in eps_list:
            a0, a1 = sharding.shard_of(q[0], rank, world, e)
            wb = max(wb, P.sfd_weak_distance_range_workspace(nF, rule, q, R, a0, a1, e, ext))
    else:
        wb = max(P.sfd_weak_distance_workspace(nF, rule, q, R, e, ext) for e in eps_list)
    work = torch.empty(wb, dtype=torch.uint8, device=dev)
    flush = torch.empty(512 << 20, dtype=torch.uint8, device=dev)
    Vj = None
    if c["jitter"]:   # config 4: the jitter is an input (workloads.jitter_vertices), applied to the device mesh
        V0, F0 = P.sfd_mesh_icosphere(level)
        Vj = torch.as_tensor(workloads.jitter_vertices(V0.cpu().numpy(), F0.cpu().numpy(), *c["jitter"]), device=dev)

    lib = P.binding._lib

    def distance(Vin, eps, s):
        if sharded:
            return sharding.weak_distance_sharded(Vin, F, rule, s, R, q, eps, work=work)
        return P.sfd_weak_distance(Vin, F, rule, s, R, q, eps, work=work)

    def step(results=None, direct_ev=None):
        rc = lib.sfd_mesh_icosphere(level, V.data_ptr(), F.data_ptr(), mesh_work.data_ptr(), mesh_work.numel(),
                                    C.c_void_p(stream.cuda_stream))
        assert rc == 0, P.binding._lib.sfd_last_error()
        Vin = Vj if Vj is not None else V
        for eps in eps_list:
            if eps == 0.0 and direct_ev is not None:
                direct_ev[0].record(stream)
            for s in c["s"]:
                d, I = distance(Vin, eps, s)
                if results is not None:
                    results[(eps, s)] = (d, I)
                    for name, ms in P.sfd_last_stage_times():
                        stage_ms.setdefault((eps, name), []).append(ms)
            if eps == 0.0 and direct_ev is not None:
                direct_ev[1].record(stream)

    stage_ms = {}
    sampler = ClockSampler(local)          # started before the warm-up so that it is sampling by the timed region
    for _ in range(max(args.warmup, 3)):
        step()
    torch.cuda.synchronize()
    P.sfd_set_profiling(True)
    results = {}
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    dev_ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    l0 = P.sfd_launch_count()
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for i in range(args.steps):
        flush.zero_()                      # evict L2 between timed steps (outside the event pair)
        ev[i][0].record(stream)
        step(results, dev_ev[i])
        ev[i][1].record(stream)
    torch.cuda.synchronize()
    t1 = time.perf_counter()
    if world > 1:
        dist.barrier()
    clocks = sampler.stop(t0, t1)
    launches = (P.sfd_launch_count() - l0) // args.steps
    # stage attribution of the NUFFT evaluations: a pass after the timed region with every stage on one stream
    Vin = Vj if Vj is not None else V
    for eps in eps_list:
        if eps > 0:
            for s in c["s"]:
                st = serial_stage_times(P, lambda: distance(Vin, eps, s), max(args.steps, 2))
                for name in [k for k in stage_ms if k[0] == eps]:
                    del stage_ms[name]
                for name, v in st.items():
                    stage_ms[(eps, name)] = v
    P.sfd_set_profiling(False)
    step_ms = [a.elapsed_time(b) for a, b in ev]
    direct_ms = [a.elapsed_time(b) for a, b in dev_ev] if 0.0 in eps_list else []
    total_ms = sum(step_ms)
    del work, flush
    torch.cuda.empty_cache()
    return dict(P=P, torch=torch, dist=dist, world=world, rank=rank, dev=dev, c=c, level=level, J=J, K=K, q=q,
                eps_list=eps_list, total_ms=total_ms, step_ms=step_ms, direct_ms=direct_ms, results=results,
                stage_ms=stage_ms, clocks=clocks, launches=launches, V=V, F=F, Vj=Vj, nV=nV, nF=nF, ext=ext,
                sharded=sharded, sharding=sharding)


def run_paper(args):
    """The paper's Fig. 4 workloads on its own variant: icosphere level N, 64-point rule, lattice M at
    xi_max = 5, transform tolerance 1e-7; timed region as in the paper = atoms + transform (the paper leaves the
    pointwise operations and the reduction out; here the deconvolution is folded into the reduction, so the reduction
    is inside the timed region too)."""
    import torch
    import paper_2304_06340_b200 as P
    torch.cuda.set_device(0)
    N, M, paper_gpu_s, paper_cpu_s = (7, 128, 0.94, 5.06) if args.workload == "fig4a" else (5, 416, 1.44, 6.42)
    V, F = P.sfd_mesh_icosphere(N)
    fp32 = args.precision == "fp32"
    if fp32:
        P.sfd_set_grid_precision(32)
    work = torch.empty(P.sfd_weak_distance_lattice_workspace(F.shape[0], 64, M, 5.0, 1e-7, 1.0), dtype=torch.uint8,
                       device="cuda")
    for _ in range(max(args.warmup, 3)):
        P.sfd_weak_distance_lattice(V, F, 64, -10.0, 5.0, M, 1e-7, work=work)
    P.sfd_set_profiling(True)
    tot, reg, stages = [], [], {}
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    launches0 = P.sfd_launch_count()
    for a, b in ev:
        a.record()
        d, I = P.sfd_weak_distance_lattice(V, F, 64, -10.0, 5.0, M, 1e-7, work=work)
        b.record()
        st = dict(P.sfd_last_stage_times())
        for k, v in st.items():
            stages.setdefault(k, []).append(v)
        # the paper's timed region: atoms + transform.  When the library folds the transform's last step (deconvolution)
        # into the reduction there is no separate "post" stage and the whole reduction is counted as well.
        skip = ("freq_nodes", "reduce") if "post" in st else ("freq_nodes",)
        reg.append(sum(v for k, v in st.items() if k not in skip))
    torch.cuda.synchronize()
    P.sfd_set_profiling(False)
    if fp32:
        P.sfd_set_grid_precision(64)
    tot = [a.elapsed_time(b) for a, b in ev]
    J, K = F.shape[0] * 64, (M + 1) ** 3
    sec = float(np.mean(reg)) * 1e-3
    launches = (P.sfd_launch_count() - launches0) // args.steps
    # which transform the library ran: the paper's type-1 (no interpolation stage) or the type-3 fallback
    transform = "type-3" if "interp" in stages else "type-1"
    line = {"metric": "seconds per evaluation: atoms + Fourier transform on the lattice (paper Fig. 4, P:244); includes the "
                      "norm's reduction, into which the deconvolution is folded",
            "value": sec, "unit": "s", "n_gpus": 1, "steps": args.steps, "warmup": max(args.warmup, 3),
            "ms_per_step": float(np.mean(tot)), "higher_is_better": False, "scaling": "weak",
            "vs_baseline": sec / paper_gpu_s, "dtype": "f32" if fp32 else "f64", "data": "synthetic",
            "config": {"workload": f"paper Fig. 4({'a' if args.workload == 'fig4a' else 'b'}): icosphere N={N}, 64-pt "
                                   f"rule, J={J} atoms; lattice M={M}, xi_max=5, K={K}; transform eps 1e-7 ({transform} NUFFT, "
                                   f"{'fp32 grids' if fp32 else 'fp64'})",
                       "paper": {"gpu_s": paper_gpu_s, "gpu": "RTX A6000, NUFFT in fp32", "cpu_s": paper_cpu_s,
                                 "cpu": "Apple M1 Max, 10 cores"}},
            "stage_ms": {k: float(np.mean(v)) for k, v in stages.items()},
            "whole_evaluation_ms": float(np.mean(tot)), "norm_H-10": d, "gpu_launches": int(launches)}
    print(json.dumps(line))
    return 0


def run_exact(args):
    """Direct summation of the exact triangle transform (eq. 2.19) on the workloads the paper quotes from the prior
    art [38]: "10 sec on NVIDIA Tesla V100 for 100 000 triangles (N ~ 6) and M = 100" and "roughly 0.1 sec for 80
    triangles (N = 1) and M = 400".  Frequencies: the paper's lattice at xi_max = 5, resident in HBM."""
    import torch
    import paper_2304_06340_b200 as P
    torch.cuda.set_device(0)
    N, M, paper_s = (6, 100, 10.0) if args.workload == "exact_a" else (1, 400, 0.1)
    V, F = P.sfd_mesh_icosphere(N)
    xi, _ = P.sfd_lattice_nodes_device(M, 5.0)
    nF, K = F.shape[0], xi.shape[0]
    for _ in range(max(args.warmup, 3)):
        out = P.sfd_exact_ft(V, F, xi)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    launches0 = P.sfd_launch_count()
    for a, b in ev:
        a.record()
        out = P.sfd_exact_ft(V, F, xi)
        b.record()
    torch.cuda.synchronize()
    launches = (P.sfd_launch_count() - launches0) // args.steps
    ms = float(np.mean([a.elapsed_time(b) for a, b in ev]))
    pairs = float(nF) * float(K)
    line = {"metric": "triangle x frequency pairs per second, exact-formula direct summation (P:128 eq. 2.19, P:244)",
            "value": pairs / (ms * 1e-3), "unit": "pairs/s", "n_gpus": 1, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": ms, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"icosphere N={N} ({nF} triangles) x lattice M={M}, xi_max=5 ({K} frequencies), "
                                   f"{pairs:.3g} pairs", "paper_quote": {"seconds": paper_s, "gpu": "Tesla V100, code of [38]",
                                                                         "note": "another machine and code: context only"}},
            "seconds": ms * 1e-3, "checksum": float(out.abs().sum().item()), "gpu_launches": int(launches)}
    print(json.dumps(line))
    return 0


def run_simulated_ranks(args):
    """One GPU, N shards one after the other: each shard's device time for the distances of `--config` (what each rank of
    a sharded N-GPU run would spend before the 16-byte all-reduce) and the sum of the partial I against the unsharded I."""
    import torch
    import paper_2304_06340_b200 as P
    from paper_2304_06340_b200 import sharding
    torch.cuda.set_device(0)
    n = args.simulate_ranks
    c, level, J, K = workload(args.config)
    q = (c["n_r"], c["n_theta"], c["n_phi"])
    V, F = P.sfd_mesh_icosphere(level)
    ext = 1.0
    if c["jitter"]:
        V = torch.as_tensor(workloads.jitter_vertices(V.cpu().numpy(), F.cpu().numpy(), *c["jitter"]), device="cuda")
        ext = 1.01
    s = c["s"][0]
    rows = []
    for eps in (c["eps"] if args.config != 2 else (0.0, 1e-9)):
        full, _, _, _ = time_distances(P, torch, args.config, level, [eps], [s], max(2, args.steps))
        shard_ms, I_sum = [], 0.0
        for r in range(n):
            a0, a1 = sharding.shard_of(q[0], r, n, eps)
            wb = P.sfd_weak_distance_range_workspace(F.shape[0], c["rule"], q, c["R"], a0, a1, eps, ext)
            work = torch.empty(max(wb, 256), dtype=torch.uint8, device="cuda")
            ms = []
            for it in range(1 + max(2, args.steps)):
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record()
                pair = P.sfd_weak_distance_range(V, F, c["rule"], s, c["R"], q, a0, a1, eps, work=work)
                e1.record()
                torch.cuda.synchronize()
                if it:
                    ms.append(e0.elapsed_time(e1))
            shard_ms.append({"rank": r, "shells": [a0, a1], "ms": float(np.median(ms))})
            I_sum += float(pair.sum())
            del work
            torch.cuda.empty_cache()
        I_full = full[(eps, s)]["I"]
        rows.append({"eps": eps, "s": s, "ms_1gpu": full[(eps, s)]["ms"], "shards": shard_ms,
                     "ms_max_shard": max(x["ms"] for x in shard_ms),
                     "speedup_bound": full[(eps, s)]["ms"] / max(x["ms"] for x in shard_ms),
                     "rel_dI_sum_of_shards": abs(I_sum - I_full) / I_full})
    print(json.dumps({"kind": "simulated_ranks", "n_ranks": n, "config": config_dict(args.config, n, "sharded"),
                      "note": "shards evaluated one after the other on ONE GPU; the all-reduce (16 B) is not included",
                      "distances": rows}))
    return 0


def main():
    args = parse_args()
    if args.impl == "reference":
        return run_reference(args)
    if args.workload != "config":
        return run_exact(args) if args.workload.startswith("exact") else run_paper(args)
    if args.simulate_ranks > 0:
        return run_simulated_ranks(args)
    r = run_sfd(args)
    P, torch, dist = r["P"], r["torch"], r["dist"]
    c, J, q = r["c"], r["J"], r["q"]
    # frequency nodes the library actually evaluates per distance: the xi_3 >= 0 half of the rule with doubled weights
    # (include/sfd.h sfd_weak_distance; exact for a real measure).  Every count below -- pairs, flops, bytes -- uses it.
    K = P.sfd_weak_distance_targets(q)
    world, rank = r["world"], r["rank"]
    n_sms = torch.cuda.get_device_properties(r["dev"]).multi_processor_count

    torch.cuda.empty_cache()   # the host-buffer calls allocate from the CUDA pool: hand torch's cached blocks back
    # ---- e2e: the same step through the host-buffer entry point (pinned host mesh in, distance out) ----------
    Vh = (r["Vj"] if r["Vj"] is not None else r["V"]).cpu().pin_memory()
    Fh = r["F"].cpu().pin_memory()
    Vn, Fn = Vh.numpy(), Fh.numpy()

    def e2e_step():
        for eps in r["eps_list"]:
            for s in c["s"]:
                P.sfd_weak_distance_host(Vn, Fn, c["rule"], s, c["R"], q, eps)

    if r["sharded"]:
        # sharded: the host-buffer entry point would evaluate the whole rule on every rank; the end-to-end step is the
        # mesh copied from pinned host memory to each rank's GPU, the rank's shard, the all-reduce, the result read back
        sharding = r["sharding"]

        def e2e_step():   # noqa: F811
            Vd = Vh.to(r["dev"], non_blocking=True)
            Fd = Fh.to(r["dev"], non_blocking=True)
            for eps in r["eps_list"]:
                for s in c["s"]:
                    sharding.weak_distance_sharded(Vd, Fd, c["rule"], s, c["R"], q, eps)

    e2e_ms = None
    if True:
        for _ in range(2):
            e2e_step()
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        t0 = time.perf_counter()
        e0.record()
        for _ in range(args.steps):
            e2e_step()
        e1.record()
        torch.cuda.synchronize()
        e2e_ms = max(e0.elapsed_time(e1), (time.perf_counter() - t0) * 1e3)   # host-blocking calls: take the wall clock
        P.sfd_release_cache()

    t = torch.tensor([r["total_ms"], e2e_ms or 0.0, sum(r["direct_ms"])], dtype=torch.float64, device=r["dev"])
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    total_ms, e2e_ms, direct_total_ms = float(t[0]), (float(t[1]) if e2e_ms is not None else None), float(t[2])
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return 0

    # pairs the step computes: the direct-sum evaluations only (one per s); times the replicas in replica mode
    n_direct = len(c["s"]) if 0.0 in r["eps_list"] else 0
    copies = world if (world > 1 and not r["sharded"]) else 1
    pairs_per_step = n_direct * J * K * copies
    ms_per_step = total_ms / args.steps
    n_dist = len(r["eps_list"]) * len(c["s"])

    # ---- per-stage device times (CUDA events recorded by the library on the launching stream) -------------------
    stages = {}
    for (eps, name), v in r["stage_ms"].items():
        stages.setdefault("direct" if eps == 0.0 else f"nufft_{eps:g}", {})[name] = float(np.mean(v))
    ms_dist = {k: sum(v.values()) for k, v in stages.items()}
    equivalent = {k: J * K / (v * 1e-3) for k, v in ms_dist.items() if k != "direct"}

    if n_direct:
        value = pairs_per_step / (ms_per_step * 1e-3)
        metric, unit = METRIC, UNIT
    else:
        # configs 3-5 run no direct sum: nothing is computed pair by pair.  The line then reports BASELINE.json's other
        # metric, ms per H^{-s} distance evaluation (median over the step's distances)
        value = ms_per_step / n_dist
        metric, unit = "ms per H^{-s} distance evaluation (type-3 NUFFT)", "ms"

    # ---- roofline of the dominant kernel ----------------------------------------------------------------------
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except OSError:
        pass
    hbm_peak, hbm_src = (peaks["hbm_gbs"], "MEASURED_PEAKS.json") if "hbm_gbs" in peaks else (6650.0, "fallback")
    fp64_tf, _ = probe_fp64(torch.cuda.current_stream().cuda_stream)
    sm_mhz = r["clocks"].get("sm_mhz") or 1965.0
    roofline, extra = None, []
    wl_tag = f"config{args.config}"
    if "direct" in stages:
        dms = stages["direct"]["direct_sum"]
        kpl = K   # nodes per launch: rank 0's shells in sharded mode
        if r["sharded"]:
            a0, a1 = r["sharding"].shard_of(q[0], 0, world, 0.0)
            kpl = K * (a1 - a0) // q[0]
        ach = FLOPS_PER_PAIR * J * kpl / (dms * 1e-3) * 1e-12
        roofline = {"kernel": "direct_sum_kernel", "bound": "alu", "achieved": ach, "peak": fp64_tf, "unit": "TFLOP/s",
                    "frac": ach / fp64_tf,
                    # dram read + write bytes of one launch from the committed ncu --set full capture (profiles/traffic.csv)
                    "traffic": measured_traffic("direct_sum_kernel", wl_tag),
                    "peak_source": "measured live by bench_probe.cu (dependency-free DFMA loop on all SMs)",
                    "peak_derived": 2 * FP64_LANES_PER_SM * n_sms * sm_mhz * 1e6 * 1e-12,
                    "pipe_frac": (DFMA_PER_PAIR + DMUL_DADD_PER_PAIR) * J * kpl / (dms * 1e-3) / (fp64_tf * 1e12 / 2),
                    "ms_per_launch": dms, "pairs_per_s": J * kpl / (dms * 1e-3),
                    "flops_per_pair": FLOPS_PER_PAIR, "algorithmic_flops": FLOPS_PER_PAIR * J * kpl}
    if not r["sharded"]:
        for eps in r["eps_list"]:
            if eps == 0.0:
                continue
            extra += nufft_rooflines(P, c, J, K, eps, stages[f"nufft_{eps:g}"], r["ext"], hbm_peak, hbm_src, sm_mhz, n_sms,
                                     wl_tag)
        if roofline is None and extra:
            roofline = dict(max(extra, key=lambda e: e["ms_per_launch"]))
            roofline["traffic"] = measured_traffic(roofline["kernel"], wl_tag)

    mode = "single" if world == 1 else ("sharded" if r["sharded"] else "replicas")
    line = {"metric": metric, "value": value, "unit": unit, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": ms_per_step, "higher_is_better": bool(n_direct),
            "scaling": "strong" if r["sharded"] else "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": config_dict(args.config, world, mode),
            "clocks": r["clocks"],
            "ms_per_step_best": float(min(r["step_ms"])), "ms_per_step_median": float(np.median(r["step_ms"])),
            "pairs_computed_per_step": pairs_per_step,
            "gpu_launches": r["launches"],
            "roofline": roofline, "roofline_nufft": extra,
            "ms_per_distance": ms_dist, "stage_ms": stages,
            "stage_ms_note": "NUFFT stages: device time per stage with every stage on one stream (a pass after the timed "
                             "region, SFD_NO_OVERLAP=1); in the timed default mode the target sort runs beside spread / fft "
                             "on a second stream, so the stages add up to more than ms_per_distance",
            "equivalent_pairs_per_s": dict(equivalent, note="NUFFT evaluations compute no pairs: J*K_evaluated / their time, "
                                                            "for comparison only, not part of `value`"),
            "distance": {f"eps={e:g},s={s:g}": d for (e, s), (d, _) in r["results"].items()}}
    if n_direct:
        line["direct_pairs_per_s"] = n_direct * J * K * copies / (direct_total_ms / args.steps * 1e-3)
    if e2e_ms is not None:
        e2e_value = pairs_per_step / (e2e_ms / args.steps * 1e-3) if n_direct else e2e_ms / args.steps / n_dist
        line["e2e"] = {"value": e2e_value, "unit": unit, "ms_per_step": e2e_ms / args.steps,
                       "h2d_bytes_per_step": (1 if r["sharded"] else n_dist) * (Vn.nbytes + Fn.nbytes),
                       "d2h_bytes_per_step": n_dist * (8 if r["sharded"] else 16),
                       "api": "sfd_weak_distance_host" if not r["sharded"] else
                              "pinned host mesh -> device, sharding.weak_distance_sharded (sfd_weak_distance_range + all-reduce)"}

    # ---- the other configurations BASELINE.json asks for in ms: config 3 (the level-6 distance) and config 5 at level 8 -
    if world == 1 and args.config == 2 and not args.no_extras:
        # (config, level, repetitions, single-precision grids): the last entry is config 3 at eps 1e-6 with the grids
        # in single precision (S:8(f) NEXT-4, the setting the paper ran its GPU NUFFT in)
        for cfg_id, lvl, reps, f32 in ((3, None, 3, False), (5, 8, 2, False), (3, None, 3, True)):
            cc = workloads.CONFIGS[cfg_id]
            eps_x = [e for e in cc["eps"] if e >= 1e-6] if f32 else list(cc["eps"])
            try:
                P.sfd_set_grid_precision(32 if f32 else 64)
                res, ext, Jx, _ = time_distances(P, torch, cfg_id, lvl, eps_x, [cc["s"][-1]], reps)
            except Exception as ex:   # e.g. not enough free memory for config 5 next to another process
                line.setdefault("extras_unavailable", {})[f"config{cfg_id}"] = str(ex)[:200]
                continue
            finally:
                P.sfd_set_grid_precision(64)
            Kx = k_evaluated(cc)
            for (eps, s), v in res.items():
                tag = f"config{cfg_id}" + (f"_L{lvl}" if lvl is not None else "") + f"_eps{eps:g}" + ("_fp32grids" if f32 else "")
                if f32:   # (the roofline entries' byte counts are fp64's: not listed for this variant)
                    line["ms_per_distance"][tag] = v["ms"]
                    line["stage_ms"][tag] = v["stage_ms"]
                    line["distance"][f"{tag},s={s:g}"] = v["distance"]
                    continue
                line["ms_per_distance"][tag] = v["ms"]
                line["stage_ms"][tag] = v["stage_ms"]
                line["distance"][f"{tag},s={s:g}"] = v["distance"]
                line["equivalent_pairs_per_s"][tag] = Jx * Kx / (v["ms"] * 1e-3)
                line["roofline_nufft"] += nufft_rooflines(P, cc, Jx, Kx, eps, v["stage_ms"], ext, hbm_peak, hbm_src, sm_mhz,
                                                          n_sms, tag)
    elif world == 1 and args.config == 5:
        # BASELINE.json config 5: "reports distance vs h (quadratic-rate check) and throughput per level": one line per
        # level and s, then the summary line (level 8) below
        prev = {}
        for lvl in range(9):
            res, ext, Jx, _ = time_distances(P, torch, 5, lvl, [1e-10], list(c["s"]), 2)
            Vl, Fl = P.sfd_mesh_icosphere(lvl)
            h = workloads.mean_edge_length(Vl.cpu().numpy(), Fl.cpu().numpy())
            for (eps, s), v in res.items():
                row = {"kind": "config5_level", "level": lvl, "s": s, "eps": eps, "J": Jx, "K_evaluated": K,
                       "mean_edge_h": h, "distance": v["distance"], "ms_per_distance": v["ms"],
                       "equivalent_pairs_per_s": Jx * K / (v["ms"] * 1e-3), "stage_ms": v["stage_ms"]}
                if s in prev:
                    row["log2_ratio_to_previous_level"] = float(np.log2(prev[s] / v["distance"]))
                prev[s] = v["distance"]
                print(json.dumps(row))
    if not args.no_cpu_baseline and world == 1:
        v, ms, cores, sample, _ = oracle_sample(args.config, args.cpu_seconds)
        line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample,
                                "ms": ms}
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
