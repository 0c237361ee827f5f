#!/usr/bin/env python
"""bench.py — headline benchmark of BASELINE.json: edges/s and structures/s for cutoff (6 A) +
KNN (k=12) graph generation on a batch of 4096 synthetic crystals (configs[2]), one B200.

A "step" is one pass of the whole hot path over the batch: mg_cutoff_graph then mg_knn_graph
through the C ABI, inputs resident in HBM.  `value` = (cutoff edges + KNN edges) * steps / time.
Between steps the outputs rotate over several buffer sets whose total size exceeds the L2, so
the edge writes really go to HBM.  `--impl reference` times the FP64 CPU oracle instead.
See DESIGN.md "Measurement" for the roofline arithmetic.
"""
from __future__ import annotations

import argparse
import ctypes
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from workloads import crystals as C  # noqa: E402

R_C, K_NN, N_STRUCT = 6.0, 12, 4096
FP32_LANES_PER_SM = 128
INSTR_PER_CANDIDATE = 7          # 3 FADD + 1 FMUL + 2 FFMA + 1 FSETP
BYTES_PER_EDGE = 23              # src 4 + dst 4 + offset 3 + vec 12


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            p = json.load(f)
        return float(p["hbm_gbs"]), float(p.get("sm_max_mhz", 1965.0)), "measured"
    return 6650.0, 1965.0, "fallback"


def box_candidates(batch, r_c):
    """C = sum_s N_s^2 prod_a (2 ceil(r_c/h_a) + 1): the search box BASELINE.json's north_star
    defines (workload statistic; plain numpy, no library code)."""
    A = batch.lattice.astype(np.float64)
    V = np.abs(np.linalg.det(A))
    h = np.stack([V / np.linalg.norm(np.cross(A[:, (a + 1) % 3], A[:, (a + 2) % 3]), axis=1)
                  for a in range(3)], axis=1)
    n = np.diff(batch.struct_ptr).astype(np.float64)
    if np.isscalar(r_c):
        r = np.full(A.shape[0], float(r_c))
    else:
        r = np.asarray(r_c, np.float64)
    cells = np.prod(2.0 * np.ceil(r[:, None] / h) + 1.0, axis=1)
    return float(np.sum(n * n * cells))


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.samples, self.reasons, self.stop_flag = index, [], set(), False
        self.max_mhz = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
        except Exception:
            self.nv = None

    def run(self):
        if self.nv is None:
            return
        nv = self.nv
        names = {"hw_slowdown": getattr(nv, "nvmlClocksThrottleReasonHwSlowdown", 0x8),
                 "hw_thermal_slowdown": getattr(nv, "nvmlClocksThrottleReasonHwThermalSlowdown", 0x40),
                 "sw_thermal_slowdown": getattr(nv, "nvmlClocksThrottleReasonSwThermalSlowdown", 0x20),
                 "sw_power_cap": getattr(nv, "nvmlClocksThrottleReasonSwPowerCap", 0x4)}
        while not self.stop_flag:
            try:
                self.samples.append(int(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                bits = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
                for k, v in names.items():
                    if bits & v:
                        self.reasons.add(k)
            except Exception:
                pass
            time.sleep(0.002)

    def result(self):
        self.stop_flag = True
        self.join(timeout=2)
        med = float(np.median(self.samples)) if self.samples else None
        return {"sm_mhz": med, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(self.samples)}


def run_reference(args, rank, world):
    """The FP64 oracle, as it stands, on the host cores (rank 0 only)."""
    if rank != 0:
        return
    import oracle
    sample_struct = 1024
    b = C.config_batch(2, n_struct=sample_struct)
    oracle.build()
    for _ in range(args.warmup):
        oracle.cutoff_graph(b.pos, b.lattice, b.struct_ptr, R_C)
    t0 = time.perf_counter()
    edges = 0
    for _ in range(args.steps):
        gc = oracle.cutoff_graph(b.pos, b.lattice, b.struct_ptr, R_C)
        gk = oracle.knn_graph(b.pos, b.lattice, b.struct_ptr, K_NN)
        edges += gc["n_edges"] + gk["n_edges"]
    dt = time.perf_counter() - t0
    val = edges / dt
    line = {"impl": "reference", "metric": "edges_per_s", "value": val, "unit": "edges/s", "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "structures_per_s": sample_struct * args.steps / dt,
            "config": {"workload": f"BASELINE configs[2]: cutoff {R_C} A + KNN k={K_NN}; each step a "
                                   f"{sample_struct}-structure prefix of the 4096-crystal batch"},
            "cpu_baseline": {"value": val, "unit": "edges/s", "cores": oracle.num_threads(), "kind": "oracle",
                             "sample": f"{sample_struct}-structure prefix, {args.steps} steps"},
            "e2e": {"value": val, "unit": "edges/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))


def run_gpu(args, rank, world, local_rank):
    import torch
    import paper_2307_05380_b200 as mg

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the graph kernels have no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)
    ctx = mg.Context(local_rank)
    lib = mg._lib()
    batch = C.config_batch(2, seed=rank)            # weak scaling: every rank has its own 4096 crystals
    pos, lat, ptr = mg.to_device(batch, dev)
    S, n_atoms = batch.n_struct, batch.n_atoms
    ctx.mg_reserve(S, n_atoms)
    e_cut = ctx.mg_cutoff_count(pos, lat, ptr, R_C)
    e_knn = K_NN * n_atoms
    bytes_cut = BYTES_PER_EDGE * e_cut + 4 * (n_atoms + 1) + 12 * n_atoms + 36 * S + 4 * (S + 1)
    bytes_knn = (BYTES_PER_EDGE + 4) * e_knn + 4 * (n_atoms + 1) + 12 * n_atoms + 36 * S + 4 * (S + 1)
    n_sets = max(2, int(np.ceil(2.2 * 126e6 / (bytes_cut + bytes_knn))))
    cut_sets = [mg.Edges.allocate(n_atoms, e_cut, dev) for _ in range(n_sets)]
    knn_sets = [mg.Edges.allocate(n_atoms, e_knn, dev, dist=True) for _ in range(n_sets)]
    cut_c = [ctypes.byref(e._c()) for e in cut_sets]
    knn_c = [ctypes.byref(e._c()) for e in knn_sets]
    h = ctx._h
    p_pos, p_lat, p_ptr = (ctypes.c_void_p(t.data_ptr()) for t in (pos, lat, ptr))
    st = ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)
    rc32 = ctypes.c_float(R_C)

    def cutoff(i):
        r = lib.mg_cutoff_graph(h, p_pos, p_lat, p_ptr, S, n_atoms, rc32, cut_c[i % n_sets], st)
        assert r == 0, r

    def knn(i):
        r = lib.mg_knn_graph(h, p_pos, p_lat, p_ptr, S, n_atoms, K_NN, knn_c[i % n_sets], st)
        assert r == 0, r

    for i in range(max(args.warmup, 3)):
        cutoff(i)
        knn(i)
    assert ctx.mg_check() == 0, "device status after warm-up"
    assert int(cut_sets[0].n_edges.item()) == e_cut and int(knn_sets[0].n_edges.item()) == e_knn

    K = args.steps
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(2 * K + 1)]
    ev_begin, ev_end = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    launches0 = ctx.mg_launch_count()
    sampler = ClockSampler(local_rank)
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    sampler.start()
    # timed region: K steps back to back, one event on each side (an event between two calls would
    # keep the next call's first kernel from being launched behind the previous call's last one)
    ev_begin.record()
    for i in range(K):
        cutoff(i)
        knn(i)
    ev_end.record()
    torch.cuda.synchronize()
    if dist is not None:
        dist.barrier()
    clocks = sampler.result()
    launches = ctx.mg_launch_count() - launches0
    total_ms = ev_begin.elapsed_time(ev_end)
    # per-call split: the same steps again with an event after every call (not part of `value`)
    ev[0].record()
    for i in range(K):
        cutoff(i)
        ev[2 * i + 1].record()
        knn(i)
        ev[2 * i + 2].record()
    torch.cuda.synchronize()
    cut_ms = sum(ev[2 * i].elapsed_time(ev[2 * i + 1]) for i in range(K)) / K
    knn_ms = sum(ev[2 * i + 1].elapsed_time(ev[2 * i + 2]) for i in range(K)) / K
    assert ctx.mg_check() == 0, "device status after the timed region"
    edges_rank = float(e_cut + e_knn)
    if dist is not None:
        t = torch.tensor([total_ms], device=dev, dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        total_ms = float(t.item())
        e = torch.tensor([edges_rank, float(S)], device=dev, dtype=torch.float64)
        dist.all_reduce(e, op=dist.ReduceOp.SUM)
        edges_all, structs_all = float(e[0].item()), float(e[1].item())
    else:
        edges_all, structs_all = edges_rank, float(S)
    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    # ---- per-kernel durations: the same steps again with the library's CUDA events (on the launching
    # stream) around every kernel; outside the timed region so that the headline carries no event cost
    ctx.mg_set_profile(True)
    for i in range(K):
        cutoff(i)
        knn(i)
    prof = ctx.mg_profile_read()
    ctx.mg_set_profile(False)
    emit_us, count_us, prep_us, knnk_us = (prof[n]["ms"] * 1e3 for n in ("emit", "count", "prep", "knn"))

    hbm_gbs, sm_mhz, peak_kind = measured_peaks()
    sms = torch.cuda.get_device_properties(dev).multi_processor_count
    fp32_rate = sms * FP32_LANES_PER_SM * sm_mhz * 1e6         # lane-instructions / s
    c_cut = box_candidates(batch, R_C)
    kn = knn_sets[(K - 1) % n_sets]
    dk = kn.dist.view(n_atoms, K_NN)[:, K_NN - 1].cpu().numpy().astype(np.float64)
    nz = np.diff(batch.struct_ptr) > 0
    dmax = np.zeros(S)
    dmax[nz] = np.maximum.reduceat(dk, batch.struct_ptr[:-1][nz])
    c_knn = box_candidates(batch, np.maximum(dmax, 1e-6))
    t_cut = {"hbm_us": bytes_cut / (hbm_gbs * 1e9) * 1e6, "fp32_us": c_cut * INSTR_PER_CANDIDATE / fp32_rate * 1e6}
    t_knn = {"hbm_us": bytes_knn / (hbm_gbs * 1e9) * 1e6, "fp32_us": c_knn * INSTR_PER_CANDIDATE / fp32_rate * 1e6}
    roof_cut, roof_knn = max(t_cut.values()), max(t_knn.values())
    kernel_us = {"mg_cut_prep_kernel": prep_us, "mg_cutoff_count_kernel": count_us,
                 "mg_cutoff_emit_kernel": emit_us, "mg_knn_pairs_kernel": knnk_us}
    traffic_all = {}
    tpath = os.path.join(ROOT, "profiles", "traffic.json")
    if os.path.exists(tpath):
        with open(tpath) as f:
            traffic_all = json.load(f)
    # the `roofline` object describes the DOMINANT kernel of the step (largest mean duration); the per-call
    # fractions are in `roofline_model`, the other kernels' in `roofline_kernels`
    def kernel_roofline(name):
        us = kernel_us[name]
        if name == "mg_knn_pairs_kernel":        # FP32-pipe bound: C_knn candidates x 7 lane-instructions
            ach = c_knn * INSTR_PER_CANDIDATE / (us * 1e-6)
            return {"bound": "alu", "achieved": ach / 1e12, "peak": fp32_rate / 1e12, "unit": "T lane-instr/s",
                    "frac": ach / fp32_rate, "kernel": name, "us": us,
                    "peak_kind": f"derived: {sms} SMs x {FP32_LANES_PER_SM} FP32 lanes x {sm_mhz:.0f} MHz (DESIGN.md 5.3)",
                    "algorithmic_lane_instr": c_knn * INSTR_PER_CANDIDATE,
                    "traffic": traffic_all.get(name + "_dram_bytes_per_launch")}
        if name == "mg_cutoff_count_kernel":     # FP32-pipe bound: the box candidates of the cutoff call
            ach = c_cut * INSTR_PER_CANDIDATE / (us * 1e-6)
            return {"bound": "alu", "achieved": ach / 1e12, "peak": fp32_rate / 1e12, "unit": "T lane-instr/s",
                    "frac": ach / fp32_rate, "kernel": name, "us": us,
                    "peak_kind": f"derived: {sms} SMs x {FP32_LANES_PER_SM} FP32 lanes x {sm_mhz:.0f} MHz (DESIGN.md 5.3)",
                    "algorithmic_lane_instr": c_cut * INSTR_PER_CANDIDATE,
                    "traffic": traffic_all.get(name + "_dram_bytes_per_launch")}
        ach = bytes_cut / (us * 1e-6) / 1e9      # the emit kernel moves the cutoff call's algorithmic bytes
        return {"bound": "hbm", "achieved": ach, "peak": hbm_gbs, "unit": "GB/s", "frac": ach / hbm_gbs,
                "kernel": name, "us": us, "peak_kind": peak_kind, "algorithmic_bytes": bytes_cut,
                "traffic": traffic_all.get(name + "_dram_bytes_per_launch")}

    graph_kernels = [k for k in kernel_us if k != "mg_cut_prep_kernel" and kernel_us[k] > 0]
    dominant = max(graph_kernels, key=lambda k: kernel_us[k])
    roofline = kernel_roofline(dominant)
    roofline_kernels = {k: kernel_roofline(k) for k in graph_kernels if k != dominant}

    # ---- end to end through the host-buffer C ABI (pinned host memory, copies inside the call)
    e2e_steps = max(3, min(K, 10))
    hp = [torch.from_numpy(a).pin_memory() for a in (batch.pos, batch.lattice, batch.struct_ptr)]

    def host_edges(cap, with_dist):
        t = dict(row_ptr=torch.empty(n_atoms + 1, dtype=torch.int32).pin_memory(),
                 src=torch.empty(cap, dtype=torch.int32).pin_memory(),
                 dst=torch.empty(cap, dtype=torch.int32).pin_memory(),
                 offset=torch.empty((cap, 3), dtype=torch.int8).pin_memory(),
                 vec=torch.empty((cap, 3), dtype=torch.float32).pin_memory(),
                 dist=torch.empty(cap, dtype=torch.float32).pin_memory() if with_dist else None,
                 n_edges=torch.zeros(1, dtype=torch.int64).pin_memory())
        c = mg._Edges(t["row_ptr"].data_ptr(), t["src"].data_ptr(), t["dst"].data_ptr(), t["offset"].data_ptr(),
                      t["vec"].data_ptr(), t["dist"].data_ptr() if with_dist else None, cap, t["n_edges"].data_ptr())
        return t, c

    hc, hc_c = host_edges(e_cut, False)
    hk, hk_c = host_edges(e_knn, False)
    hargs = [ctypes.c_void_p(t.data_ptr()) for t in hp]

    def e2e_step():
        r1 = lib.mg_cutoff_graph_host(h, hargs[0], hargs[1], hargs[2], S, n_atoms, rc32, ctypes.byref(hc_c))
        r2 = lib.mg_knn_graph_host(h, hargs[0], hargs[1], hargs[2], S, n_atoms, K_NN, ctypes.byref(hk_c))
        assert r1 == 0 and r2 == 0, (r1, r2)

    e2e_step()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        e2e_step()
    torch.cuda.synchronize()
    e2e_s = (time.perf_counter() - t0) / e2e_steps
    assert int(hc["n_edges"][0]) == e_cut and int(hk["n_edges"][0]) == e_knn
    in_bytes = 2 * (12 * n_atoms + 36 * S + 4 * (S + 1))
    out_bytes = BYTES_PER_EDGE * (e_cut + e_knn) + 2 * (4 * (n_atoms + 1) + 8 + 4)

    # ---- the oracle on the host cores, bounded sample (N=1 only)
    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        import oracle
        reps = 8
        oracle.build()
        t0 = time.perf_counter()
        ne = 0
        for _ in range(reps):
            ne += oracle.cutoff_graph(batch.pos, batch.lattice, batch.struct_ptr, R_C)["n_edges"]
            ne += oracle.knn_graph(batch.pos, batch.lattice, batch.struct_ptr, K_NN)["n_edges"]
        dt = time.perf_counter() - t0
        cpu = {"value": ne / dt, "unit": "edges/s", "cores": oracle.num_threads(), "kind": "oracle",
               "sample": f"the full {S}-structure batch, cutoff + KNN, {reps} repetitions ({dt:.1f} s)",
               "structures_per_s": S * reps / dt}
        # the other configs, one repetition each (SURVEY 8(d) "Oracle timed beside it")
        try:
            b3c = C.config_batch(3, n_struct=4)
            t0 = time.perf_counter()
            g3 = oracle.cutoff_graph(b3c.pos, b3c.lattice, b3c.struct_ptr, 8.0)
            cpu["config3_cutoff"] = {"s": time.perf_counter() - t0, "edges": int(g3["n_edges"]), "sample": "4 of the 16 supercells"}
            b4c = C.config_batch(4)
            t0 = time.perf_counter()
            for _ in range(3):
                oracle.knn_graph(b4c.pos, b4c.lattice, b4c.struct_ptr, 24)
            cpu["config4_knn24_s_per_step"] = (time.perf_counter() - t0) / 3
            os.environ["OMP_NUM_THREADS"] = "1"
            import subprocess
            one = subprocess.run([sys.executable, "-c",
                                  "import sys, time; sys.path.insert(0, %r)\n"
                                  "import oracle; from workloads import crystals as C\n"
                                  "b = C.config_batch(2, n_struct=512); t0 = time.perf_counter()\n"
                                  "e = oracle.cutoff_graph(b.pos, b.lattice, b.struct_ptr, %f)['n_edges'] + "
                                  "oracle.knn_graph(b.pos, b.lattice, b.struct_ptr, %d)['n_edges']\n"
                                  "print(e / (time.perf_counter() - t0))" % (ROOT, R_C, K_NN)],
                                 capture_output=True, text=True, env=dict(os.environ, OMP_NUM_THREADS="1"))
            del os.environ["OMP_NUM_THREADS"]
            if one.returncode == 0:
                cpu["single_thread_edges_per_s"] = float(one.stdout.strip().splitlines()[-1])
                cpu["single_thread_sample"] = "512-structure prefix of configs[2], cutoff + KNN, OMP_NUM_THREADS=1"
        except Exception as ex:      # the extra timings are context; the headline baseline stands without them
            cpu["extra_error"] = repr(ex)

    # ---- config 4: dynamic geometry, mg_update_graph KNN k=24 on 1024 skewed crystals, 100 steps of
    # a pre-generated trajectory resident on the device (per-step latency, BASELINE.json metric)
    upd = None
    if world == 1 and not args.no_update:
        k4, n_steps = 24, 100
        b4 = C.config_batch(4)
        traj = list(C.walk(b4, n_steps, seed=0))
        tpos = torch.from_numpy(np.stack([t.pos for t in traj])).to(dev)
        tlat = torch.from_numpy(np.stack([t.lattice for t in traj])).to(dev)
        ptr4 = torch.from_numpy(b4.struct_ptr).to(dev)
        graph = ctx.mg_graph_create(mg.MG_KIND_KNN, ptr4, b4.n_atoms, k=k4)
        out4 = mg.Edges.allocate(b4.n_atoms, k4 * b4.n_atoms, dev, dist=True)
        c4 = ctypes.byref(out4._c())
        # (device addresses of every step's inputs, taken before the timed loops: the host does nothing per step but
        # the call itself)
        ppos = [ctypes.c_void_p(tpos[i].data_ptr()) for i in range(n_steps)]
        plat = [ctypes.c_void_p(tlat[i].data_ptr()) for i in range(n_steps)]
        for i in range(5):
            lib.mg_update_graph(h, graph._h, ppos[i], plat[i], c4, st)
        torch.cuda.synchronize()
        # pass 1: the 100 steps enqueued back to back, one pair of events around them
        ea, eb = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ea.record()
        for i in range(n_steps):
            r = lib.mg_update_graph(h, graph._h, ppos[i], plat[i], c4, st)
            assert r == 0, r
        eb.record()
        torch.cuda.synchronize()
        assert ctx.mg_check() == 0, "device status after the update steps"
        piped_us = ea.elapsed_time(eb) * 1e3 / n_steps
        # pass 2: the same steps with an event after each one (the distribution; an event between two calls keeps the
        # next call's first kernel from overlapping the tail of the last one)
        ev4 = [torch.cuda.Event(enable_timing=True) for _ in range(n_steps + 1)]
        ev4[0].record()
        for i in range(n_steps):
            r = lib.mg_update_graph(h, graph._h, ppos[i], plat[i], c4, st)
            assert r == 0, r
            ev4[i + 1].record()
        torch.cuda.synchronize()
        assert ctx.mg_check() == 0, "device status after the update steps"
        lat_us = np.array([ev4[i].elapsed_time(ev4[i + 1]) * 1e3 for i in range(n_steps)])
        upd = {"workload": f"BASELINE configs[4]: mg_update_graph KNN k={k4}, {b4.n_struct} skewed crystals, "
                           f"{b4.n_atoms} atoms, {n_steps} steps enqueued back to back",
               "us_per_step": {"mean": float(piped_us), "how": "one event pair around the 100 steps"},
               "us_per_step_events": {"mean": float(lat_us.mean()), "median": float(np.median(lat_us)),
                                      "max": float(lat_us.max()), "how": "an event after every step"},
               "edges_per_s": float(k4 * b4.n_atoms / (piped_us * 1e-6))}
        graph.close()

    # ---- pure-write bandwidth of this GPU, measured here: a fill of as many bytes as the cutoff call emits
    # (the measured HBM peak is a COPY, read + write bytes; an edge list is written only)
    write_only = None
    if world == 1 and not args.no_latency:
        fb = [torch.empty(int(bytes_cut), dtype=torch.int8, device=dev) for _ in range(n_sets)]
        for i in range(4):
            fb[i % n_sets].fill_(1)
        torch.cuda.synchronize()
        f0, f1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        f0.record()
        for i in range(50):
            fb[i % n_sets].fill_(1)
        f1.record()
        torch.cuda.synchronize()
        fill_us = f0.elapsed_time(f1) * 1e3 / 50
        write_only = {"bytes": int(bytes_cut), "fill_us": fill_us, "gbs": bytes_cut / fill_us / 1e3,
                      "note": "torch.Tensor.fill_ of the cutoff call's algorithmic bytes, buffers rotating beyond L2"}
        del fb

    # ---- single-call latency: one call, one synchronisation (median / p99 over 200 calls each)
    latency = None
    if world == 1 and not args.no_latency:
        def call_latency(fn, n=200):
            ts = []
            for i in range(n):
                torch.cuda.synchronize()
                t0 = time.perf_counter()
                fn(i)
                torch.cuda.synchronize()
                ts.append((time.perf_counter() - t0) * 1e6)
            a = np.array(ts)
            return {"median_us": float(np.median(a)), "p99_us": float(np.percentile(a, 99))}
        latency = {"cutoff": call_latency(cutoff), "knn": call_latency(knn), "how": "host clock around call + cudaDeviceSynchronize"}

    # ---- the other configs and calls (one leg each; events around `reps` back-to-back calls)
    legs = {}
    if world == 1 and not args.no_legs:
        def timed(fn, reps=50, warm=3):
            for i in range(warm):
                fn(i)
            torch.cuda.synchronize()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            for i in range(reps):
                fn(i)
            b.record()
            torch.cuda.synchronize()
            assert ctx.mg_check() == 0
            return a.elapsed_time(b) * 1e3 / reps

        # BASELINE configs[3]: cutoff 8 A on 16 supercells of 500-2000 atoms
        b3 = C.config_batch(3)
        p3, l3, s3 = mg.to_device(b3, dev)
        e3 = ctx.mg_cutoff_count(p3, l3, s3, 8.0)
        o3 = [mg.Edges.allocate(b3.n_atoms, e3, dev) for _ in range(2)]
        us3 = timed(lambda i: ctx.mg_cutoff_graph(p3, l3, s3, 8.0, o3[i % 2]), reps=20)
        n3 = np.diff(b3.struct_ptr).astype(np.float64)
        bytes3 = BYTES_PER_EDGE * e3 + 4 * (b3.n_atoms + 1) + 12 * b3.n_atoms + 40 * b3.n_struct
        roof3 = max(float(np.sum(n3 * n3)) * INSTR_PER_CANDIDATE / fp32_rate * 1e6, bytes3 / (hbm_gbs * 1e9) * 1e6)
        legs["config3_cutoff"] = {"workload": f"BASELINE configs[3]: cutoff 8 A, {b3.n_struct} supercells, {b3.n_atoms} atoms",
                                  "us_per_call": us3, "edges": int(e3), "edges_per_s": e3 / (us3 * 1e-6),
                                  "candidates_min_image": float(np.sum(n3 * n3)), "roof_us": roof3, "frac": roof3 / us3}
        # ... and KNN on the same supercells (knn_bins.cu: a warp per row through the cell list)
        ok3 = [mg.Edges.allocate(b3.n_atoms, K_NN * b3.n_atoms, dev, dist=True) for _ in range(2)]
        us3k = timed(lambda i: ctx.mg_knn_graph(p3, l3, s3, K_NN, ok3[i % 2]), reps=20)
        legs["config3_knn12"] = {"workload": f"KNN k={K_NN} on the supercells of BASELINE configs[3]", "us_per_call": us3k,
                                 "edges": int(K_NN * b3.n_atoms), "edges_per_s": K_NN * b3.n_atoms / (us3k * 1e-6)}
        del o3, ok3

        # the shape of the paper's Table 1: batch of 256 cells of up to 64 atoms
        bp = C.paper_scale_batch(256)
        pp, lp, sp_ = mg.to_device(bp, dev)
        tab = {}
        for k in (16, 32, 64):
            ok_ = mg.Edges.allocate(bp.n_atoms, k * bp.n_atoms, dev, dist=True)
            tab[f"knn{k}_ms_per_batch"] = timed(lambda i: ctx.mg_knn_graph(pp, lp, sp_, k, ok_), reps=30) * 1e-3
        for rc in (3.0, 5.0, 8.0):
            ec = ctx.mg_cutoff_count(pp, lp, sp_, rc)
            oc = mg.Edges.allocate(bp.n_atoms, ec, dev)
            tab[f"cutoff{rc:g}_ms_per_batch"] = timed(lambda i: ctx.mg_cutoff_graph(pp, lp, sp_, rc, oc), reps=30) * 1e-3
        legs["paper_scale_batch256"] = dict(tab, workload=f"256 synthetic cells of 1-64 atoms ({bp.n_atoms} atoms), the shape of the paper's "
                                            "Table 1 batch row (PAPER.md:138: 53 / 55 / 80 ms KNN, 43 / 72 / 123 ms cutoff on an RTX 8000, "
                                            "Materials Project data: context, another machine and other data)")

        # a few large structures among the small cells of the headline batch (a Materials-Project-like mix: the batch still
        # averages below 64 atoms per structure, so it takes the headline's kernels, mg_knn_row_box)
        mixed = {}
        for tag, big in (("plus_1x100_atoms", [C.supercell(7, 0, density=100 / 20.0 ** 3 / 0.9, n_lo=100, n_hi=140)]),
                         ("plus_8x900_atoms", [C.supercell(7, s_, n_lo=900, n_hi=1100) for s_ in range(8)])):
            bm = C.concat([batch, C._assemble(big)])
            pm, lm, sm_ = mg.to_device(bm, dev)
            om = mg.Edges.allocate(bm.n_atoms, K_NN * bm.n_atoms, dev, dist=True)
            mixed[tag] = {"n_atoms": int(bm.n_atoms), "knn_us_per_call": timed(lambda i: ctx.mg_knn_graph(pm, lm, sm_, K_NN, om), reps=20)}
            em = ctx.mg_cutoff_count(pm, lm, sm_, R_C)
            om = mg.Edges.allocate(bm.n_atoms, em, dev)
            mixed[tag]["cutoff_us_per_call"] = timed(lambda i: ctx.mg_cutoff_graph(pm, lm, sm_, R_C, om), reps=20)
            del om
        legs["config2_with_large_structures"] = dict(mixed, workload="BASELINE configs[2] plus one 100-140-atom / eight 900-1100-atom "
                                                     f"structures, KNN k={K_NN} and cutoff {R_C:g} A")

        # SURVEY 8(f) NEXT-1 / NEXT-2 on the headline KNN graph: symmetric graph, triplets
        kn = knn_sets[0]
        sym = mg.Edges.allocate(n_atoms, 2 * e_knn, dev, dist=True)
        us_sym = timed(lambda i: ctx.mg_symmetrize(kn, n_atoms, sym), reps=30)
        n_tri = K_NN * (K_NN - 1) * n_atoms
        # (outputs allocated once, as a caller in a loop would; the binding's convenience call allocates per call)
        tri_ptr = torch.empty(n_atoms + 1, dtype=torch.int64, device=dev)
        tri_a, tri_b = torch.empty(n_tri, dtype=torch.int32, device=dev), torch.empty(n_tri, dtype=torch.int32, device=dev)
        tri_n = torch.zeros(1, dtype=torch.int64, device=dev)
        tri_c = mg._Triplets(tri_ptr.data_ptr(), tri_a.data_ptr(), tri_b.data_ptr(), n_tri, tri_n.data_ptr())
        rp_knn = ctypes.c_void_p(kn.row_ptr.data_ptr())
        us_tri = timed(lambda i: lib.mg_triplets_graph(h, rp_knn, n_atoms, ctypes.byref(tri_c), st), reps=30)
        assert int(tri_n.item()) == n_tri
        legs["symmetrize_knn12"] = {"us_per_call": us_sym, "edges_in": int(e_knn), "edges_out": int(sym.n_edges.item())}
        legs["triplets_knn12"] = {"us_per_call": us_tri, "triplets": int(n_tri), "gbs_written": 8.0 * n_tri / us_tri / 1e3}
        # per-atom cutoffs drawn in [2, 6.5] A on the headline batch
        rad = torch.from_numpy(np.random.default_rng(0).uniform(2.0, 6.5, n_atoms).astype(np.float32)).to(dev)
        orad = mg.Edges.allocate(n_atoms, e_cut, dev)
        us_rad = timed(lambda i: ctx.mg_cutoff_graph_radii(pos, lat, ptr, rad, orad), reps=30)
        legs["cutoff_radii"] = {"us_per_call": us_rad, "edges": int(orad.n_edges.item())}

    line = {
        "metric": "edges_per_s", "value": edges_all * K / (total_ms * 1e-3), "unit": "edges/s",
        "n_gpus": world, "steps": K, "warmup": max(args.warmup, 3), "ms_per_step": total_ms / K,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
        "data": "synthetic",
        "config": {"workload": f"BASELINE configs[2]: cutoff r_c={R_C} A + KNN k={K_NN} on {S} crystals per GPU "
                               f"(N in [1,20], lengths 3-10 A, angles 60-120 deg, min distance 1 A), seed = rank",
                   "n_struct": S, "n_atoms": n_atoms, "cutoff_edges": e_cut, "knn_edges": e_knn,
                   "l2": f"outputs rotate over {n_sets} buffer sets ({n_sets * (bytes_cut + bytes_knn) / 1e6:.0f} MB "
                         f"> 126 MB L2); inputs are {12 * n_atoms + 40 * S} B"},
        "structures_per_s": structs_all * K / (total_ms * 1e-3),
        "call_us": {"cutoff": cut_ms * 1e3, "knn": knn_ms * 1e3},
        "kernel_us": kernel_us,
        "roofline": roofline,
        "roofline_kernels": roofline_kernels,
        "roofline_model": {"cutoff": dict(t_cut, candidates=c_cut, roof_us=roof_cut, frac=roof_cut / (cut_ms * 1e3)),
                           "knn": dict(t_knn, candidates=c_knn, roof_us=roof_knn, frac=roof_knn / (knn_ms * 1e3)),
                           "fp32_peak_lane_instr_per_s": fp32_rate,
                           "step_frac": (roof_cut + roof_knn) / (total_ms / K * 1e3),
                           "edge_only_floor_us": {"cutoff": e_cut * INSTR_PER_CANDIDATE / fp32_rate * 1e6,
                                                  "knn": e_knn * INSTR_PER_CANDIDATE / fp32_rate * 1e6},
                           "write_only": write_only},
        "e2e": {"value": (e_cut + e_knn) / e2e_s, "unit": "edges/s", "h2d_bytes_per_step": in_bytes,
                "d2h_bytes_per_step": out_bytes, "ms_per_step": e2e_s * 1e3, "steps": e2e_steps},
        "gpu_launches": int(launches),
        "clocks": clocks,
    }
    if upd is not None:
        line["update_graph"] = upd
    if latency is not None:
        line["latency"] = latency
    if legs:
        line["legs"] = legs
    if cpu is not None:
        line["cpu_baseline"] = cpu
    print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=300)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-update", action="store_true", help="skip the configs[4] mg_update_graph latency leg")
    ap.add_argument("--no-latency", action="store_true", help="skip the single-call latency and write-only bandwidth measurements")
    ap.add_argument("--no-legs", action="store_true", help="skip the configs[3] / paper-scale / graph-operation legs")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank, world)
        return
    run_gpu(args, rank, world, local_rank)


if __name__ == "__main__":
    main()
