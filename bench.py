#!/usr/bin/env python
"""bench.py -- hash-renderer throughput on the BASELINE.json workload (one step = one 800x800 frame through the whole
hot path a1-a11: encode, BRDF decoder, implicit ray tracer, secondary hit, recursive re-evaluation, rendering sum).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload C2|C3|C1|C3a] [--impl ours|reference]

Prints ONE JSON line (rank 0).  `value` = point-direction queries/s (device-resident inputs, CUDA events, max over
ranks); `e2e` = the same metric through hashrender_render_frame_host (pinned host buffers, H2D + D2H inside the timed
region); `roofline` = algorithmic work of the render kernel / its measured duration against the measured peak;
`cpu_baseline` = the oracle, as it stands, on a bounded pixel sample of the same workload.
`--impl reference` times the oracle alone (rank 0; other ranks exit).  See DESIGN.md "Measurement".
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import gen  # noqa: E402

METRIC = "hash-renderer point-direction queries/s (800x800 frame, direct + shadow + one-bounce indirect)"
UNIT = "queries/s"


def algorithmic_flops(cfg, evaluated=None) -> float:
    """Factored algorithmic flop count of one frame: per IRT query
    2*(3*64 + 64*64 + 64*2) = 8832; per encoded point the per-point layer-1 partial 2*D*64 and, where B runs,
    2*(D*64 + 64*64 + 64*7).  Zero padding to MMA shapes and error-compensation passes are never counted.
    `evaluated` = secondary hits whose L'_o was actually evaluated (None = all N*S_i of them, the dense count)."""
    D, H = cfg.D, cfg.hidden
    per_query = 2 * (3 * H + H * H + H * 2)
    per_point = 2 * D * H + 2 * (D * H + H * H + H * 7)
    ind = bool(cfg.flags & gen.HR_INDIRECT)
    sec = cfg.N * cfg.S_i if ind else 0
    ev = sec if evaluated is None else evaluated
    queries = cfg.N * cfg.S_d + sec + ev * cfg.S_2
    return queries * per_query + (cfg.N + ev) * per_point


def executed_queries(cfg, evaluated=None) -> int:
    ind = bool(cfg.flags & gen.HR_INDIRECT)
    sec = cfg.N * cfg.S_i if ind else 0
    ev = sec if evaluated is None else evaluated
    return cfg.N * cfg.S_d + sec + ev * cfg.S_2


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return dict(hbm=d["hbm_gbs"], tensor=d["bf16_tflops"], tensor_sustained=d.get("bf16_tflops_sustained", d["bf16_tflops"]),
                    sm_max_mhz=d.get("sm_max_mhz", 1965.0), which="measured")
    return dict(hbm=6650.0, tensor=1590.0, tensor_sustained=1400.0, sm_max_mhz=1965.0, which="fallback")


class ClockSampler:
    """Samples nvidia-smi clocks + throttle reasons while the timed region runs (B200_PROFILING.md clocks line).  The nvidia-smi
    loop is started before the warm-up (it needs ~0.2 s to come up) and every row is stamped on arrival; stop() keeps the rows
    that arrived between begin() and end()."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.rows, self.proc = index, [], None
        self.t0, self.t1, self.window = None, None, "timed region"

    def start(self):
        if self.proc:
            return
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-i", str(self.index),
                                          "-lms", "50"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), [c.strip() for c in line.split(",")]))

    def begin(self):
        self.t0 = time.time()

    def end(self, window=None):
        self.t1 = time.time()
        if window:
            self.window = window

    def in_window(self):
        return [r for (ts, r) in self.rows if len(r) >= 6 and self.t0 is not None and self.t0 <= ts <= (self.t1 or time.time()) + 0.06]

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        rows = self.in_window()
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm = [float(r[0]) for r in rows if r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in rows if r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = sorted({names[i] for r in rows for i in range(4) if r[2 + i].lower().startswith("active")})
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None, "reasons": reasons,
                "samples": len(sm), "window": self.window}


def oracle_sample(cfg, model, pix, vis_mode):
    """Times the oracle on the pixels `pix` of the workload.  Returns (seconds, queries)."""
    from oracle.oracle import Oracle
    fr = gen.make_frame(cfg, model["env"], pix)
    o = Oracle.from_gen(cfg, model, vis_mode=vis_mode)
    sec = (fr["dir_s"], fr["pdf_s"]) if cfg.flags & gen.HR_INDIRECT else None
    ter = (fr["dir_t"], fr["pdf_t"]) if cfg.flags & gen.HR_INDIRECT else None
    t0 = time.perf_counter()
    o.render_frame(fr["x"], fr["wo"], (fr["dir_d"], fr["pdf_d"]), sec, ter, flags=cfg.flags)
    dt = time.perf_counter() - t0
    return dt, len(pix) * cfg.queries // cfg.N


def _oracle_worker(job):
    name, pix, vis_mode = job
    cfg = gen.make_config(name)
    model = gen.make_model(cfg)
    return oracle_sample(cfg, model, pix, vis_mode)


def oracle_all_cores(cfg, pix, vis_mode, procs):
    """The same oracle, one single-threaded instance per host core over disjoint pixel ranges.  Each worker rebuilds the
    model from the seed (untimed) and times only its render; the rate is total queries / slowest worker."""
    import multiprocessing as mp
    parts = [p for p in np.array_split(pix, procs) if len(p)]
    with mp.get_context("spawn").Pool(len(parts)) as pool:
        res = pool.map(_oracle_worker, [(cfg.name, p, vis_mode) for p in parts])
    return max(r[0] for r in res), sum(r[1] for r in res), len(parts)


def sample_pixels(cfg, n, seed=1234):
    return np.sort(np.random.default_rng(seed).choice(cfg.N, n, replace=False))


def run_reference(args, cfg):
    """--impl reference: the oracle, as it stands, single-threaded on the host; each step = a bounded pixel sample."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    model = gen.make_model(cfg)
    npx = args.ref_pixels
    for _ in range(args.warmup):
        oracle_sample(cfg, model, sample_pixels(cfg, max(npx // 8, 8)), args.vis_mode)
    tot, q = 0.0, 0
    for k in range(args.steps):
        dt, qq = oracle_sample(cfg, model, sample_pixels(cfg, npx, seed=1234 + k), args.vis_mode)
        tot += dt; q += qq
    val = q / tot
    sample = f"{npx} seeded pixels of the {cfg.name} frame per step ({npx * cfg.queries // cfg.N} queries), {args.steps} steps"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": tot / args.steps * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_name(cfg), "sample": sample},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


def ncu_record(key):
    """Counters of the dominant kernel copied from the ncu --set full capture named in the record (profiles/ncu_metrics.json;
    `capture` says which report).  They are NOT measured by this run: traffic = dram__bytes_read.sum + dram__bytes_write.sum
    per launch, issue_slots_busy / tensor_pipe_active in % of active cycles, warp_inst = smsp__inst_executed.sum."""
    pth = os.path.join(ROOT, "profiles", "ncu_metrics.json")
    if not os.path.exists(pth):
        return None
    return json.load(open(pth)).get(key)


_GATHER = None


def gather_model():
    """The L1 roofline of the hash-grid gathers, measured live with hashrender_probe_gather (fully divergent loads from a 32 MiB,
    L2-resident table, 160 KiB of shared memory requested as the render kernels do): an SM passes one missing 32-byte sector per
    `c_sector + c_load` cycles when every load has a sector of its own, and every further load of the same sector costs `c_load`.
    cycles per point = c_sector * sectors + c_load * loads."""
    global _GATHER
    if _GATHER is None:
        from paper_2409_10327_b200.binding import probe_gather
        rows = {}
        for name, (w, grp) in {"4B x1": (4, 1), "4B x2 per sector": (4, 2), "4B x4 per sector": (4, 4), "4B x8 per sector": (4, 8),
                               "8B x1": (8, 1), "32B x1": (32, 1)}.items():
            per_cycle, per_s = probe_gather(32 << 20, w, grp, 160 << 10)
            rows[name] = {"loads_per_cycle_per_sm": per_cycle, "loads_per_s": per_s}
        c1 = 1.0 / rows["4B x1"]["loads_per_cycle_per_sm"]              # cycles per load = per sector
        c2 = 2.0 / rows["4B x2 per sector"]["loads_per_cycle_per_sm"]   # cycles per sector with two loads in it
        c_load = c2 - c1
        _GATHER = {"probe": rows, "c_sector": c1 - c_load, "c_load": c_load,
                   "l1_hit": probe_gather(16 << 10, 4, 1, 160 << 10)[0]}
    return _GATHER


def gather_counts(levels, cell_major, rows_per_sector):
    """(32-byte sectors, load instructions) one point's encode touches: a cell-major level is one sector and one 256-bit load
    (fp16 rows, 8 per sector) or two and two (fp32 rows, 4 per sector); any other level is 4 x-pairs, and the two rows of a pair --
    rows s and s ^ m with m = cx ^ (cx + 1) = 1, 3, 7, ... -- share a sector unless m >= rows_per_sector, which happens for one
    cell in rows_per_sector.  Loads of such a level: 8 one-row loads for fp32 rows; for fp16 rows one two-row load per pair plus a
    one-row load of the neighbour when cx is odd (hr_device.cuh gather8_h2): 6 on average.  The sector count is checked against a
    count over the oracle's indices in tests/test_gen_recipe.py."""
    per_entry = 1 if rows_per_sector == 8 else 2
    sectors = cell_major * per_entry + (levels - cell_major) * 4 * (1 + 1.0 / rows_per_sector)
    loads = cell_major * per_entry + (levels - cell_major) * (6 if rows_per_sector == 8 else 8)
    return sectors, loads


def gather_floor(n_points, levels, cell_major, rows_per_sector, sm_mhz, num_sms=148):
    """L1 floor of the encode of n_points: cell-major levels cost one sector and one load (fp16) or two and two (fp32 rows),
    the others 8 loads in 4 x-pairs, each pair in one sector unless it straddles a sector boundary."""
    gm = gather_model()
    sectors, loads = gather_counts(levels, cell_major, rows_per_sector)
    cyc = gm["c_sector"] * sectors + gm["c_load"] * loads
    ms = n_points * cyc / num_sms / (sm_mhz * 1e3)
    return {"sectors_per_point": sectors, "loads_per_point": loads, "c_sector": gm["c_sector"], "c_load": gm["c_load"],
            "cycles_per_point": cyc, "floor_ms": ms, "sm_mhz": sm_mhz,
            "probe_loads_per_cycle_per_sm": gm["probe"]["4B x1"]["loads_per_cycle_per_sm"],
            "probe_loads_per_s": gm["probe"]["4B x1"]["loads_per_s"]}


C4_ALG_BYTES = 16 * 8 * 4 + 24 + 8      # per point: 128 gathers x one fp16 pair + position / direction in + (v, t) out


def measure_c4(log2_T, Ns, steps, vis_mode, peaks, clock_index=None):
    """encode + IRT (hashrender_trace, encode fused, 1 direction / point; BASELINE.json configs[4]) at one table size for the
    point counts `Ns`.  One row per N, each with its own clock record when clock_index is given."""
    import torch
    from paper_2409_10327_b200 import DirSet, HashRenderer
    dev = torch.device("cuda", torch.cuda.current_device())
    cfg = gen.make_config("C4", log2_T=log2_T, N=max(Ns))
    model = gen.make_model(cfg)
    r = HashRenderer.from_gen(cfg, model, vis_mode=vis_mode, max_points=max(Ns))
    del model
    g = torch.Generator(device=dev); g.manual_seed(4)
    x = torch.rand((max(Ns), 3), device=dev, generator=g)
    d = torch.randn((max(Ns), 1, 3), device=dev, generator=g); d = (d / d.norm(dim=2, keepdim=True)).contiguous()
    pdf = torch.ones((max(Ns), 1), device=dev)
    vis = torch.empty((max(Ns), 1), device=dev); t = torch.empty((max(Ns), 1), device=dev)
    rows = []
    for N in Ns:
        ds = DirSet(d[:N], pdf[:N])
        clocks = ClockSampler(clock_index) if clock_index is not None else None
        if clocks:
            clocks.start()
        for _ in range(3):
            r.trace(x[:N], None, ds, vis, None, t, N=N)
        torch.cuda.synchronize()
        if clocks:
            clocks.begin()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(steps):
            r.trace(x[:N], None, ds, vis, None, t, N=N)
        e1.record(); torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / steps
        clk = None
        if clocks:
            clocks.end()
            if len(clocks.in_window()) < 8:          # short timed region: sample over an untimed continuation of the same launches
                t_end = time.time() + 1.0
                while time.time() < t_end:
                    for _ in range(4):
                        r.trace(x[:N], None, ds, vis, None, t, N=N)
                    torch.cuda.synchronize()
                clocks.end("timed region + 1 s untimed continuation of the same launches")
            clk = clocks.stop()
        useful = N * 16 * 8 * 4            # bytes actually used: 8 corners x 16 levels x one fp16 pair
        alg = N * C4_ALG_BYTES
        path = r.last_path()
        rec = ncu_record(f"C4:T{log2_T}:N{N.bit_length() - 1}:{path}") or {}
        roof = {"bound": "hbm", "achieved": alg / (ms * 1e-3) / 1e9, "peak": peaks["hbm"], "unit": "GB/s",
                "frac": alg / (ms * 1e-3) / 1e9 / peaks["hbm"], "traffic": rec.get("traffic"), "kernel": "k_trace_wg", "kernel_ms": ms,
                "algorithmic_bytes_per_point": C4_ALG_BYTES, "peak_source": f"MEASURED_PEAKS.json hbm_gbs ({peaks['which']})",
                "capture": rec.get("capture"),
                "note": "a 4-byte gather moves a 32-byte sector, so sector traffic is up to 8x the algorithmic bytes; tables <= 32 MiB "
                        "(T <= 2^19) are L2-resident and the bound there is the L1/L2 gather rate, not HBM"}
        if rec.get("traffic"):
            roof["traffic_GBps"] = rec["traffic"] / (ms * 1e-3) / 1e9
            roof["traffic_frac_of_peak"] = roof["traffic_GBps"] / peaks["hbm"]
        nblock, dev_bytes = r.table_layout()
        mhz = (clk or {}).get("sm_mhz") or 1900.0
        l1 = gather_floor(N, 16, nblock, 8, mhz)
        l1["frac"] = l1["floor_ms"] / ms
        l1["note"] = ("floor of the encode's gathers alone at the L1 sector-request rate measured by hashrender_probe_gather; it binds while "
                      "the table is L2-resident (T <= 2^20), HBM traffic binds beyond")
        roof["l1_gather"] = l1
        roof["cell_major_levels"] = nblock
        roof["device_table_MiB"] = dev_bytes / 2 ** 20
        rows.append({"log2_T": log2_T, "table_MiB": 16 * (1 << log2_T) * 4 / 2 ** 20, "N": N, "ms": ms, "points_per_s": N / (ms * 1e-3),
                     "useful_gather_GBps": useful / (ms * 1e-3) / 1e9, "sector_GBps_upper": useful * 8 / (ms * 1e-3) / 1e9,
                     "path": path, "roofline": roof, "clocks": clk})
    r.destroy(); del x, d, pdf, vis, t
    torch.cuda.empty_cache()
    return rows


def run_c4_sweep(args):
    """BASELINE.json configs[4]: encode + IRT throughput (hashrender_trace, encode fused, 1 direction / point) over
    N = 2^20..2^26 uniform random points x T = 2^16, 2^19, 2^22, 2^24 (fp16, F=2, L=16): where the gather leaves L2."""
    import torch
    torch.cuda.set_device(0)
    peaks = load_peaks()
    gran = None
    if args.l2_fetch_granularity:
        import ctypes
        torch.zeros(1, device="cuda")
        rt = ctypes.CDLL("libcudart.so.12")
        rc = rt.cudaDeviceSetLimit(5, ctypes.c_size_t(args.l2_fetch_granularity))          # cudaLimitMaxL2FetchGranularity = 0x05
        got = ctypes.c_size_t(0)
        rt.cudaDeviceGetLimit(ctypes.byref(got), 5)
        gran = {"requested": args.l2_fetch_granularity, "rc": rc, "in_effect": got.value}
    rows = []
    Ns = [1 << 20, 1 << 22, 1 << 24] + ([1 << 26] if args.full_sweep else [])
    if args.c4_n:
        Ns = [args.c4_n]
    for log2_T in ((args.c4_log2t,) if args.c4_log2t else (16, 19, 22, 24)):
        rows += measure_c4(log2_T, Ns, args.steps, args.vis_mode, peaks, clock_index=0)
    best = max(rows, key=lambda q: q["points_per_s"])
    hb = max(rows, key=lambda q: (q["log2_T"], q["N"]))          # the HBM end of the sweep: largest table, most points
    print(json.dumps({"metric": "encode+IRT points/s (BASELINE.json configs[4] sweep)", "value": best["points_per_s"], "unit": "points/s", "n_gpus": 1,
                      "steps": args.steps, "warmup": 3, "ms_per_step": best["ms"], "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                      "dtype": "f16", "data": "synthetic", "config": {"workload": "C4 sweep: uniform random points x 1 direction, fp16 L=16 F=2",
                      "points": "generated on device (torch Philox); parity of this call at every table size of the sweep: tests/test_gpu_parity.py::test_c4_sweep_full_size_sampled_points"},
                      "l2_fetch_granularity": gran, "hbm_peak_GBps": peaks["hbm"], "clocks": hb["clocks"], "gpu_launches": args.steps, "roofline": hb["roofline"], "sweep": rows}))


def measure_gbuffer(steps, peaks, clock_index=None, cpu_rays=40):
    """The step before the path: one forward pass of the CNN direct renderer G (hashrender_gbuffer_forward; PAPER.md:68, 90-96,
    134) at the paper's shape, 100 x 100 rays -> 800 x 800 maps of x, n, a, r, mask, random-init weights.  Reports ms / frame, the
    algorithmic tensor rate (2 N Cout Cin k^2 per convolution, ONE pass: the second pass over the lo halves of the split
    activations is this implementation's cost, not algorithmic work) against the measured bf16 peak, and the float64 oracle timed
    beside it on a smaller ray array."""
    import torch
    from gen import gnet
    from paper_2409_10327_b200 import GBufferNet
    dev = torch.device("cuda", torch.cuda.current_device())
    blob = gnet.make_gnet(7)
    rays_h = gnet.make_rays(7, 100, 100)
    net = GBufferNet(blob, 100, 100)
    rays = torch.from_numpy(rays_h).to(dev)
    N = net.N
    x = torch.empty((N, 3), device=dev); brdf = torch.empty((N, 7), device=dev); mask = torch.empty((N,), device=dev, dtype=torch.uint8)
    stream = torch.cuda.current_stream().cuda_stream
    clocks = ClockSampler(clock_index) if clock_index is not None else None
    if clocks:
        clocks.start()
    for _ in range(3):
        net.forward(rays, x, brdf, mask, stream=stream)
    torch.cuda.synchronize()
    l0 = net.launch_count()
    if clocks:
        clocks.begin()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(steps):
        net.forward(rays, x, brdf, mask, stream=stream)
    e1.record(); torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / steps
    launches = (net.launch_count() - l0) // steps
    clk = None
    if clocks:
        clocks.end()
        if len(clocks.in_window()) < 8:
            t_end = time.time() + 1.0
            while time.time() < t_end:
                for _ in range(8):
                    net.forward(rays, x, brdf, mask, stream=stream)
                torch.cuda.synchronize()
            clocks.end("timed region + 1 s untimed continuation of the same launches")
        clk = clocks.stop()
    # the same 77 launches captured once into a CUDA graph and replayed (every call of the library only enqueues on the caller's
    # stream: no allocation, no synchronisation, so the pass is capturable as it stands)
    graph_ms = None
    try:
        side = torch.cuda.Stream()
        side.wait_stream(torch.cuda.current_stream())
        gr = torch.cuda.CUDAGraph()
        with torch.cuda.graph(gr, stream=side):
            net.forward(rays, x, brdf, mask, stream=side.cuda_stream)
        for _ in range(3):
            gr.replay()
        torch.cuda.synchronize()
        e0.record()
        for _ in range(steps):
            gr.replay()
        e1.record(); torch.cuda.synchronize()
        graph_ms = e0.elapsed_time(e1) / steps
        del gr
    except Exception as exc:                                           # report, never hide
        graph_ms = f"capture failed: {exc}"
    # end to end: the ray map travels host -> device, the maps come back
    hr_ = torch.from_numpy(rays_h).pin_memory()
    hx = torch.empty((N, 3)).pin_memory(); hb = torch.empty((N, 7)).pin_memory()
    def e2e():
        rd = hr_.to(dev, non_blocking=True)
        net.forward(rd, x, brdf, mask, stream=stream)
        hx.copy_(x, non_blocking=True); hb.copy_(brdf, non_blocking=True)
        torch.cuda.synchronize()
    e2e()
    e0.record()
    for _ in range(3):
        e2e()
    e1.record(); torch.cuda.synchronize()
    e2e_ms = e0.elapsed_time(e1) / 3
    flops = net.flops()
    ach = flops / (ms * 1e-3) / 1e12
    rec = ncu_record("G:k_gconv") or {}
    out = {"workload": "G: CNN direct renderer forward, 100x100 rays -> 800x800 maps (width 256, 28 residual layers, SR blocks 128/64/32; "
                       "PAPER.md:134), random-init weights", "ms_per_frame": ms, "kernels_per_frame": launches, "finite": bool(torch.isfinite(x).all()),
           "cuda_graph_replay_ms_per_frame": graph_ms,
           "e2e_ms_per_frame": e2e_ms, "h2d_bytes_per_step": int(rays_h.nbytes), "d2h_bytes_per_step": int(N * 40),
           "paper_context": "Model Op. 4.3-5.8 ms on an A100 (PAPER.md:185-193, trained weights; context only)",
           "roofline": {"bound": "tensor", "achieved": ach, "peak": peaks["tensor_sustained"], "unit": "TFLOP/s", "frac": ach / peaks["tensor_sustained"],
                        "algorithmic_flops_per_frame": flops, "kernel": "k_gconv (35 launches per frame) + element-wise stages",
                        "traffic": rec.get("traffic"), "capture": rec.get("capture"),
                        "peak_source": f"MEASURED_PEAKS.json bf16_tflops_sustained ({peaks['which']})",
                        "note": "143 GFLOP per frame is 0.1 ms of tensor time: the pass is bound by the 77 dependent launches (every instance "
                                "norm needs the whole image's statistics) and by the fp32 element-wise stages, not by the MMAs"},
           "clocks": clk}
    net.destroy()
    # the oracle on a smaller ray array (cost is linear in the pixel count)
    from oracle import gnet_oracle as G
    t0 = time.perf_counter()
    G.forward(blob, gnet.make_rays(7, cpu_rays, cpu_rays))
    dt = time.perf_counter() - t0
    out["cpu_baseline"] = {"value": dt * (100.0 / cpu_rays) ** 2 * 1e3, "unit": "ms/frame (extrapolated)", "kind": "oracle", "cores": os.cpu_count(),
                           "sample": f"{cpu_rays}x{cpu_rays} rays -> {8 * cpu_rays}x{8 * cpu_rays} maps in {dt:.1f} s (numpy float64, BLAS threads)"}
    return out


def workload_name(cfg):
    ind = f" + {cfg.S_i} secondary x {cfg.S_2} tertiary (one-bounce indirect)" if cfg.flags & gen.HR_INDIRECT else ""
    return (f"{cfg.name}: 800x800 = {cfg.N} primary points, {cfg.S_d} direct directions{ind}; L={cfg.L} F={cfg.F} T=2^{cfg.log2_T} "
            f"{cfg.table_dtype} tables, {cfg.mlp_dtype} MLPs (BASELINE.json configs[{ {'C1': 1, 'C2': 2, 'C3': 3, 'C3a': 3}.get(cfg.name, '?') }])")


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="C2", choices=["C1", "C2", "C3", "C3a", "C4", "G", "probe"])
    ap.add_argument("--full-sweep", action="store_true", help="C4: include 2^26 points")
    ap.add_argument("--c4-log2t", type=int, default=0, help="C4: only this table size (for profiling one point of the sweep)")
    ap.add_argument("--c4-n", type=int, default=0, help="C4: only this many points")
    ap.add_argument("--l2-fetch-granularity", type=int, default=0, help="probe: cudaDeviceSetLimit(cudaLimitMaxL2FetchGranularity, n) in this "
                    "process before the measurement (32 / 64 / 128 bytes; 0 = leave the driver default)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--vis-mode", type=int, default=1, help="1 = hard visibility (paper-faithful), 0 = soft")
    ap.add_argument("--e2e-steps", type=int, default=3)
    ap.add_argument("--cpu-pixels", type=int, default=2048, help="pixels of the frame the cpu_baseline leg evaluates")
    ap.add_argument("--ref-pixels", type=int, default=256, help="pixels per step for --impl reference")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-cpu-all-cores", action="store_true", help="skip the all-host-cores oracle leg")
    ap.add_argument("--also", default="C1,C3,C4,G", help="comma-separated workloads measured briefly and reported under `also` ('' = none); "
                    "C4 = the T = 2^19 and T = 2^24 points of the sweep at 2^24 points; G = the CNN direct renderer forward")
    ap.add_argument("--compact", action="store_true", help="headline with the default API flags (zero-weight secondary rays skipped) "
                    "instead of HR_DENSE")
    ap.add_argument("--no-extra", action="store_true", help="skip the `also` measurements")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 0)
    if args.workload == "G" and args.impl != "reference":
        import torch
        torch.cuda.set_device(0)
        g = measure_gbuffer(args.steps, load_peaks(), clock_index=0)
        print(json.dumps({"metric": "G forward ms/frame (100x100 rays -> 800x800 maps)", "value": g["ms_per_frame"], "unit": "ms", "n_gpus": 1,
                          "steps": args.steps, "warmup": 3, "ms_per_step": g["ms_per_frame"], "higher_is_better": False, "scaling": "weak",
                          "vs_baseline": None, "dtype": "f16x2 (fp16 hi+lo split activations, fp32 accumulate)", "data": "synthetic",
                          "config": {"workload": g["workload"]}, "clocks": g["clocks"], "gpu_launches": g["kernels_per_frame"] * args.steps,
                          "roofline": g["roofline"], "cpu_baseline": g["cpu_baseline"],
                          "e2e": {"value": g["e2e_ms_per_frame"], "unit": "ms", "h2d_bytes_per_step": g["h2d_bytes_per_step"],
                                  "d2h_bytes_per_step": g["d2h_bytes_per_step"]}}))
        return
    if args.workload == "probe" and args.impl != "reference":
        import torch
        torch.cuda.set_device(0)
        torch.zeros(1, device="cuda")
        gm = gather_model()
        print(json.dumps({"metric": "divergent-gather rate of an SM's L1 (hashrender_probe_gather)", "value": gm["probe"]["4B x1"]["loads_per_s"],
                          "unit": "loads/s", "n_gpus": 1, "higher_is_better": True, "data": "synthetic",
                          "config": {"workload": "512 threads per SM, 8 independent pseudo-random slots in flight per thread, 32 MiB table "
                                                 "(L2-resident), 160 KiB dynamic shared memory"},
                          "probe": gm["probe"], "c_sector": gm["c_sector"], "c_load": gm["c_load"], "l1_hit_loads_per_cycle_per_sm": gm["l1_hit"]}))
        return
    cfg = gen.make_config("C2" if args.workload in ("G", "probe") else args.workload)
    if args.impl == "reference":
        return run_reference(args, gen.make_config("C2") if args.workload == "C4" else cfg)
    if args.workload == "C4":
        return run_c4_sweep(args)

    import torch
    import torch.distributed as dist
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (no CPU fallback exists)"
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    dev = torch.device("cuda", local)

    from paper_2409_10327_b200 import DirSet, HashRenderer
    from paper_2409_10327_b200 import dist as hd

    def measure(cfg, steps, warmup, e2e_steps, clocks, dense=True, sampled=False):
        model = gen.make_model(cfg)
        fr = gen.make_frame(cfg, model["env"])
        r = HashRenderer.from_gen(cfg, model, vis_mode=args.vis_mode)
        up = lambda a: torch.from_numpy(a).to(dev)
        r.set_env(up(model["env"]))
        indirect = bool(cfg.flags & gen.HR_INDIRECT)
        x, wo = up(fr["x"]), up(fr["wo"])
        d = DirSet(up(fr["dir_d"]), up(fr["pdf_d"]))
        s = DirSet(up(fr["dir_s"]), up(fr["pdf_s"])) if indirect else None
        t = DirSet(up(fr["dir_t"]), up(fr["pdf_t"])) if indirect else None
        flags = cfg.flags | (gen.HR_DENSE if dense else 0)
        frame = r.make_frame(x, wo, d, s, t, flags=flags)
        rgb = torch.empty((cfg.N, 3), device=dev)
        stream = torch.cuda.current_stream().cuda_stream
        if clocks:
            clocks.start()
        for _ in range(warmup):
            r.render_frame(frame, rgb, stream)
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        r.stats(reset=True)
        l0 = r.launch_count()
        if clocks:
            clocks.begin()
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(steps + 1)]
        torch.cuda.synchronize()
        ev[0].record()
        for k in range(steps):
            r.render_frame(frame, rgb, stream)
            ev[k + 1].record()
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        launches = r.launch_count() - l0
        traced, evaluated = r.stats()
        clk = None
        if clocks:
            clocks.end()
            if len(clocks.in_window()) < 8:
                # a short timed region (K x ~20 ms) sees only a few 50 ms samples: keep sampling over an UNTIMED continuation of the
                # same launches, so the reported clocks and throttle reasons are those of this kernel under sustained load
                t_end = time.time() + 1.0
                while time.time() < t_end:
                    for _ in range(4):
                        r.render_frame(frame, rgb, stream)
                    torch.cuda.synchronize()
                clocks.end("timed region + 1 s untimed continuation of the same launches")
            clk = clocks.stop()
        total_ms = ev[0].elapsed_time(ev[-1])
        per = [ev[k].elapsed_time(ev[k + 1]) for k in range(steps)]
        total_ms = hd.max_over_ranks(total_ms, dev)
        assert torch.isfinite(rgb).all()
        out = dict(total_ms=total_ms, per=per, launches=launches, clk=clk, path=r.last_path(), mean_rgb=float(rgb.mean().item()),
                   traced=traced // max(steps, 1), evaluated=(evaluated // max(steps, 1)) if traced else None,
                   cell_major=r.table_layout()[0], device_table_MiB=r.table_layout()[1] / 2 ** 20)
        # end to end through the public host-buffer entry point: pinned host inputs, H2D + D2H inside the timed region
        if e2e_steps:
            pin = lambda a: torch.from_numpy(a).pin_memory().numpy()
            hx, hwo = pin(fr["x"]), pin(fr["wo"])
            hdir = DirSet(pin(fr["dir_d"]), pin(fr["pdf_d"]))
            hs = DirSet(pin(fr["dir_s"]), pin(fr["pdf_s"])) if indirect else None
            ht = DirSet(pin(fr["dir_t"]), pin(fr["pdf_t"])) if indirect else None
            hframe = r.make_frame(hx, hwo, hdir, hs, ht, flags=flags)
            hrgb = torch.empty((cfg.N, 3), dtype=torch.float32).pin_memory().numpy()
            upb, downb = r.render_frame_host(hframe, hrgb, stream)      # warm-up (allocates staging)
            torch.cuda.synchronize()
            if world > 1:
                dist.barrier()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for _ in range(e2e_steps):
                upb, downb = r.render_frame_host(hframe, hrgb, stream)
            e1.record()
            torch.cuda.synchronize()
            out.update(e2e_ms=hd.max_over_ranks(e0.elapsed_time(e1), dev) / e2e_steps, h2d=upb, d2h=downb,
                       e2e_matches=bool(np.allclose(hrgb, rgb.cpu().numpy(), rtol=1e-5, atol=1e-6)))
        # end to end with the directions generated ON the device: only x, wo travel host->device; the primary
        # BRDF is decoded (encode + decode), the direct set is the MIS light + GGX set of PAPER.md:122 (spp = S_d / 2), the
        # secondary set a stratified cosine hemisphere about the decoded normal, the tertiary set a shared stratified sphere
        if e2e_steps and sampled:
            import math
            hx, hwo = torch.from_numpy(fr["x"]).pin_memory(), torch.from_numpy(fr["wo"]).pin_memory()
            hrgb = torch.empty((cfg.N, 3), dtype=torch.float32).pin_memory()
            N = cfg.N
            feat = torch.empty((N, cfg.D), device=dev); brdf = torch.empty((N, 7), device=dev)
            dd = torch.empty((N, cfg.S_d, 3), device=dev); pd = torch.empty((N, cfg.S_d), device=dev)
            sa = int(math.isqrt(cfg.S_i)) if indirect else 0
            if indirect:
                ds_ = torch.empty((N, sa * sa, 3), device=dev); ps_ = torch.empty((N, sa * sa), device=dev)
                ta, tb = (cfg.S_2 // 2, 2) if cfg.S_2 % 2 == 0 else (cfg.S_2, 1)
                dt_ = torch.empty((ta * tb, 3), device=dev); pt_ = torch.empty((ta * tb,), device=dev)

            def sampled_frame():
                xd = hx.to(dev, non_blocking=True); wod = hwo.to(dev, non_blocking=True)
                r.encode(xd, feat, stream=stream)
                r.decode(feat, brdf, stream=stream)
                r.sample_mis(brdf, wod, cfg.S_d // 2, 2409, dd, pd, stream=stream)
                sset = tset = None
                if indirect:
                    nrm = brdf[:, :3].contiguous()
                    r.sample_stratified(nrm, N, sa, sa, 10327, ds_, ps_, stream=stream)
                    r.sample_stratified(None, 1, ta, tb, 7, dt_, pt_, stream=stream)
                    sset, tset = DirSet(ds_, ps_), DirSet(dt_, pt_)
                fq = r.make_frame(xd, wod, DirSet(dd, pd), sset, tset, flags=flags)
                r.render_frame(fq, rgb, stream)
                hrgb.copy_(rgb, non_blocking=True)
                torch.cuda.synchronize()

            sampled_frame()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for _ in range(e2e_steps):
                sampled_frame()
            e1.record()
            torch.cuda.synchronize()
            out.update(e2e_sampled_ms=e0.elapsed_time(e1) / e2e_steps, e2e_sampled_h2d=int(hx.numel() + hwo.numel()) * 4,
                       e2e_sampled_finite=bool(torch.isfinite(hrgb).all()), e2e_sampled_mean=float(hrgb.mean()))
        # the step after the path: spatial-only SVGF on the frame just rendered ("Dnsr" column of Table 3)
        if sampled and cfg.points == "scene" and cfg.N == cfg.width * cfg.width:
            Wd = cfg.width
            nimg = up(fr["n_g"]).reshape(Wd, Wd, 3); pimg = x.reshape(Wd, Wd, 3); rimg = rgb.reshape(Wd, Wd, 3)
            dout = torch.empty_like(rimg)
            for _ in range(2):
                r.denoise(rimg, nimg, pimg, (0.5, 0.5, -1.2), dout, stream=stream)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for _ in range(10):
                r.denoise(rimg, nimg, pimg, (0.5, 0.5, -1.2), dout, stream=stream)
            e1.record(); torch.cuda.synchronize()
            out.update(denoise_ms=e0.elapsed_time(e1) / 10, denoise_finite=bool(torch.isfinite(dout).all()))
        r.destroy()
        del x, wo, d, s, t, rgb
        torch.cuda.empty_cache()
        return out, model

    peaks = load_peaks()
    clocks = ClockSampler(local) if rank == 0 else None
    res, model = measure(cfg, args.steps, max(args.warmup, 3), args.e2e_steps, clocks, dense=not args.compact, sampled=world == 1)

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    ms = res["total_ms"] / args.steps
    value = world * cfg.queries / (ms * 1e-3)
    kernel_ms = float(np.mean(res["per"]))          # the step is ONE kernel launch: its duration is the step's

    def roofline(cfg, path, kernel_ms, evaluated, res=None):
        flops = algorithmic_flops(cfg, evaluated)
        ach = flops / (kernel_ms * 1e-3) / 1e12
        if path.startswith("tcgen05"):
            # the contraction's own dtype is fp16 with fp32 accumulate for BOTH tensor paths: the peak is the measured sustained
            # fp16 / bf16 rate, undivided.  (The split-precision path spends three MMA passes per product; that is this
            # implementation's cost, not a smaller roofline.)
            roof = {"bound": "tensor", "achieved": ach, "peak": peaks["tensor_sustained"], "unit": "TFLOP/s",
                    "peak_source": f"MEASURED_PEAKS.json bf16_tflops_sustained ({peaks['which']}; fp16 = bf16 rate; kernel runs back to back for the whole step)"}
        else:
            alu_peak = 148 * 128 * 2 * peaks["sm_max_mhz"] * 1e6 / 1e12
            roof = {"bound": "alu", "achieved": ach, "peak": alu_peak, "unit": "TFLOP/s",
                    "peak_source": "derived: 148 SM x 128 fp32 lanes x 2 flop x sm_max_mhz (DESIGN.md)"}
        roof["frac"] = roof["achieved"] / roof["peak"]
        if path == "tcgen05-f16x3":
            roof["frac_over_3pass"] = 3.0 * roof["frac"]       # share of the tensor pipe's time the three passes would need at peak; not `frac`
        roof["kernel"] = "k_render_wg" if path.startswith("tcgen05") else "k_render_ffma"
        roof["kernel_ms"] = kernel_ms
        roof["algorithmic_flops_per_launch"] = flops
        roof["note"] = ("the MLP contractions run on the tensor pipe, but the kernel's binding unit is the SM issue slots: per query the "
                        "fp16 pack / epilogue / shading ALU work exceeds the 64x64 MMA (DESIGN.md 6.1); see profiles/ for issue-slot "
                        "and tensor-pipe utilisation")
        rec = ncu_record(f"{cfg.name}:{path}") or {}
        roof["traffic"] = rec.get("traffic")
        for k in ("issue_slots_busy", "tensor_pipe_active", "capture"):
            roof[k] = rec.get(k)
        if rec.get("warp_inst"):                               # thread instructions per executed query, from the capture's dense frame
            roof["thread_inst_per_query"] = rec["warp_inst"] * 32 / cfg.queries
        if res is not None and path.startswith("tcgen05") and world == 1:
            # the second roofline of this kernel: the L1 sector-request rate of the encode's gathers (every primary point and every
            # evaluated secondary hit is encoded once), measured live by hashrender_probe_gather
            ind = bool(cfg.flags & gen.HR_INDIRECT)
            ev = (cfg.N * cfg.S_i if evaluated is None else evaluated) if ind else 0
            mhz = (res.get("clk") or {}).get("sm_mhz") or 1900.0
            l1 = gather_floor(cfg.N + ev, cfg.L, res["cell_major"], 8 if cfg.table_dtype == "f16" else 4, mhz)
            l1["frac"] = l1["floor_ms"] / kernel_ms
            l1["encoded_points"] = cfg.N + ev
            l1["note"] = ("time the encode's gathers alone need at the measured L1 rate for divergent loads; the kernel cannot run faster than "
                          "max(this, the issue-slot floor), and its gathers and MMA round trips overlap only partly")
            roof["l1_gather"] = l1
            roof["cell_major_levels"] = res["cell_major"]
            roof["device_table_MiB"] = res["device_table_MiB"]
        return roof

    roof = roofline(cfg, res["path"], kernel_ms, res["evaluated"], res)
    dt = {"tcgen05-f16": "f16", "tcgen05-f16x3": "f16x3 (fp16 hi+lo split operands, three tcgen05 passes, fp32 accumulate)"}.get(res["path"], "f32")
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
        "ms_per_step": ms, "ms_per_frame": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": dt, "data": "synthetic",
        "config": {"workload": workload_name(cfg), "queries_per_frame": cfg.queries, "vis_mode": "hard" if args.vis_mode else "soft",
                   "secondary_rays": ("compacted: L'_o only where its Eq. 2 weight is non-zero (PAPER.md:82-84)" if args.compact else
                                      "dense (HR_DENSE): L'_o evaluated at every secondary hit, all queries_per_frame executed"),
                   "executed_queries_per_frame": executed_queries(cfg, res["evaluated"]),
                   "path": res["path"], "l2": "per-frame inputs (2.0 GB of directions/pdfs) exceed the 126 MB L2; the hash table is "
                   "L2-resident by design", "multi_gpu": "independent frames per rank, no collective"},
        "clocks": res["clk"], "gpu_launches": res["launches"], "mean_rgb": res["mean_rgb"], "roofline": roof,
    }
    if "e2e_ms" in res:
        line["e2e"] = {"value": world * cfg.queries / (res["e2e_ms"] * 1e-3), "unit": UNIT, "ms_per_frame": res["e2e_ms"],
                       "h2d_bytes_per_step": res["h2d"], "d2h_bytes_per_step": res["d2h"], "matches_device_path": res["e2e_matches"]}
    if "e2e_sampled_ms" in res:
        line["e2e_sampled"] = {"value": cfg.queries / (res["e2e_sampled_ms"] * 1e-3), "unit": UNIT, "ms_per_frame": res["e2e_sampled_ms"],
                               "h2d_bytes_per_step": res["e2e_sampled_h2d"], "d2h_bytes_per_step": cfg.N * 12, "finite": res["e2e_sampled_finite"],
                               "mean_rgb": res["e2e_sampled_mean"],
                               "parity": "tests/test_gpu_sampler.py::test_sampled_frame_composition_matches_oracle checks this composition against the "
                                         "composition of the oracles",
                               "what": "same frame shape, but only x and wo travel: B(H(x)) is decoded and the direction sets are generated on the "
                                       "device (hashrender_encode/decode/sample_mis/sample_stratified/render_frame); PAPER.md:122, 344"}
    if "denoise_ms" in res:
        line["denoise"] = {"ms_per_frame": res["denoise_ms"], "finite": res["denoise_finite"], "kernels_per_frame": 7,
                           "what": "hashrender_denoise: spatial-only SVGF (7x7 variance estimate + five 5x5 a-trous passes) on the rendered "
                                   "800x800 frame; the paper's Table 3 lists 3.2-3.5 ms for its denoiser on an A100 (context)"}
    if world == 1 and not args.no_extra:
        # the same frame with the default API flags (zero-weight secondary rays compacted out), the other
        # BASELINE configs (C1 direct only, C3 fp16) and two points of the C4 sweep (T = 2^19 L2-resident, T = 2^24 HBM, both at
        # 2^24 points); `value` here is frame-equivalent (queries_per_frame / time), executed queries are stated
        extra = []
        if cfg.flags & gen.HR_INDIRECT:
            extra.append((cfg, args.compact))
        for nm in [w for w in args.also.split(",") if w and w != args.workload and w not in ("C4", "G")]:
            cfg2 = gen.make_config(nm)
            extra += [(cfg2, True), (cfg2, False)] if cfg2.flags & gen.HR_INDIRECT else [(cfg2, True)]
        line["also"] = []
        for c2, dense in extra:
            st = max(args.steps // 2, 3)
            r2, _ = measure(c2, st, 3, 0, ClockSampler(local), dense=dense)
            ms2 = r2["total_ms"] / st
            rf = roofline(c2, r2["path"], ms2, r2["evaluated"], r2)
            line["also"].append({"workload": workload_name(c2), "secondary_rays": "dense" if dense else "compacted", "ms_per_frame": ms2,
                                 "frame_equivalent_queries_per_s": c2.queries / (ms2 * 1e-3),
                                 "executed_queries_per_frame": executed_queries(c2, r2["evaluated"]),
                                 "executed_queries_per_s": executed_queries(c2, r2["evaluated"]) / (ms2 * 1e-3), "path": r2["path"],
                                 "mean_rgb": r2["mean_rgb"], "achieved_tflops": rf["achieved"], "roofline_frac": rf["frac"],
                                 "roofline_peak": rf["peak"], "roofline": rf, "clocks": r2["clk"]})
        if "G" in args.also.split(","):
            line["gbuffer"] = measure_gbuffer(max(args.steps, 5), peaks, clock_index=local)
        if "C4" in args.also.split(","):
            for log2_T in (19, 24):
                for row in measure_c4(log2_T, [1 << 24], max(args.steps // 2, 3), args.vis_mode, peaks, clock_index=local):
                    line["also"].append({"workload": f"C4: encode + IRT, 2^24 uniform random points x 1 direction, fp16 L=16 F=2 T=2^{log2_T} "
                                                     f"({row['table_MiB']:.0f} MiB table; BASELINE.json configs[4])", "ms": row["ms"],
                                         "points_per_s": row["points_per_s"], "path": row["path"], "roofline_frac": row["roofline"]["frac"],
                                         "roofline": row["roofline"], "clocks": row["clocks"]})
    if not args.no_cpu_baseline and world == 1:
        pix = sample_pixels(cfg, args.cpu_pixels)
        dt, q = oracle_sample(cfg, model, pix, args.vis_mode)
        line["cpu_baseline"] = {"value": q / dt, "unit": UNIT, "cores": 1, "kind": "oracle",
                                "sample": f"{len(pix)} seeded pixels of the same {cfg.name} frame ({q} queries) in {dt:.1f} s; "
                                          f"full frame extrapolates to {dt * cfg.N / len(pix):.0f} s",
                                "host_cores_available": os.cpu_count()}
        avail = len(os.sched_getaffinity(0))
        if not args.no_cpu_all_cores and avail > 1:
            procs = min(avail, 64)
            npx = min(cfg.N, max(1, args.cpu_pixels // 2) * procs)
            dta, qa, used = oracle_all_cores(cfg, sample_pixels(cfg, npx, seed=4321), args.vis_mode, procs)
            line["cpu_baseline"]["all_cores"] = {"value": qa / dta, "unit": UNIT, "cores": used,
                                                 "sample": f"{npx} seeded pixels split over {used} single-threaded oracle "
                                                           f"processes; slowest took {dta:.1f} s"}
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
