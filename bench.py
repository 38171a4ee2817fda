#!/usr/bin/env python
"""bench.py -- the hot path of liboptimus_b200 timed on B200 (contract: DESIGN.md "Measurement").

A STEP is one pass of the whole hot path over one batch of
seeded synthetic input, i.e. the fused op groups of BASELINE.json configs[1..4] back to back,
SIX kernel launches, one per group:

    C1   batched LayerNorm      64 members [2048, D_i]                      1 launch
    C2   grouped Linear+ReLU    128 members, M=4096, concat output          1 launch
    C3   split-pointwise-cat    [8192, 8192], 256 chunks, permuted          1 launch
    C4   recsys block           512 towers: LN -> Linear+ReLU -> Linear     3 launches

(configs[0] is the tiny fp32 parity case; it is launch-latency bound and is timed only as a
side figure.)  Metric: fused op-group latency, microseconds per step (BASELINE.json:metric);
per-group latency, TFLOP/s or GB/s and roofline fractions ride in "groups".

  python bench.py [--gpus N] [--steps K] [--warmup W]      product arm (CUDA, through the C ABI)
  python bench.py --impl reference ...                      CPU oracle arm (bounded row sample)

N > 1: "replicas only" -- every rank runs the same step on its own
GPU, no collective on the data path; time = max over ranks.
"""
import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import workloads as wl  # noqa: E402

BF16, F32 = wl.BF16, wl.F32
ACT_NONE, ACT_RELU = 0, 1
FULL = dict(c1_rows=2048, c1_n=64, c2_M=4096, c2_n=128, c3_rows=8192, c3_width=8192, c3_chunks=256,
            c4_B=8192, c4_n=512)
SMALL = dict(c1_rows=256, c1_n=16, c2_M=512, c2_n=16, c3_rows=512, c3_width=2048, c3_chunks=64,
             c4_B=512, c4_n=24)


NCU_SUMMARY = os.path.join(ROOT, "profiles", "r02_ncu_full_metrics.csv")
GEMM_SOURCES = ["paper_2607_02945_b200/csrc/grouped_gemm_sm100.cuh", "paper_2607_02945_b200/csrc/linear.cu",
                "paper_2607_02945_b200/csrc/sm100_ptx.h"]


def gemm_source_sha():
    import hashlib
    h = hashlib.sha256()
    for f in GEMM_SOURCES:
        with open(os.path.join(ROOT, f), "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()[:16]


def ncu_traffic_of_gemm_launches():
    """roofline.traffic: dram__bytes_read.sum + dram__bytes_write.sum of the step's three grouped-GEMM launches (C2,
    C4b, C4c), read at run time from the committed ncu summary (profiles/r02_ncu_full_metrics.csv, written by
    `bench.py --ncu-summary` from one `ncu --set full` capture of `bench.py --profile`).  The summary records the
    sha of the kernel's sources at capture time: if the sources have changed since, the figure is stale -> None."""
    import csv
    if not os.path.exists(NCU_SUMMARY):
        return None, "no ncu summary committed"
    rows = {r[0]: r[1:] for r in csv.reader(open(NCU_SUMMARY)) if r}
    if rows.get("gemm_source_sha16", ["", ""])[1] != gemm_source_sha():
        return None, "stale: %s was captured from other kernel sources" % os.path.basename(NCU_SUMMARY)
    names = rows["metric"][1:]
    total = 0.0
    for key in ("dram__bytes_read.sum", "dram__bytes_write.sum"):
        unit, vals = rows[key][0], rows[key][1:]
        scale = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}[unit]
        total += sum(float(v) * scale for n_, v in zip(names, vals) if "GEMM" in n_)
    return int(total), "profiles/%s (ncu --set full, one step)" % os.path.basename(NCU_SUMMARY)


def write_ncu_summary(rep):
    """`python bench.py --ncu-summary gpurun_out/prof_r02_full.ncu-rep > profiles/r02_ncu_full_metrics.csv` (on the
    CPU box): one column per launch of the captured step, the metrics the roofline discussion uses, and the sha of the
    grouped GEMM's sources."""
    import csv
    import subprocess
    raw = subprocess.run(["ncu", "-i", rep, "--page", "raw", "--csv"], capture_output=True, text=True, check=True).stdout
    rows = list(csv.reader(raw.splitlines()))
    hdr, units, data = rows[0], rows[1], rows[2:]
    labels = ["C1 LN", "C2 GEMM", "C3 pointwise", "C4a LN", "C4b GEMM", "C4c GEMM"]
    if len(data) != 6:          # a side-workload capture: one column per captured launch, in capture order
        labels = ["launch %d" % i for i in range(len(data))]
    keep = ["Kernel Name", "Grid Size", "Block Size", "gpu__time_duration.sum", "dram__bytes_read.sum", "dram__bytes_write.sum",
            "gpu__dram_throughput.avg.pct_of_peak_sustained_elapsed", "sm__pipe_tensor_cycles_active.avg.pct_of_peak_sustained_active",
            "sm__throughput.avg.pct_of_peak_sustained_elapsed", "smsp__issue_active.avg.pct_of_peak_sustained_active",
            "lts__throughput.avg.pct_of_peak_sustained_elapsed", "lts__t_bytes.sum", "lts__t_sectors_srcunit_tex.sum",
            "l1tex__m_xbar2l1tex_read_bytes.sum", "sm__warps_active.avg.pct_of_peak_sustained_active", "launch__registers_per_thread",
            "sm__cycles_active.avg", "sm__cycles_elapsed.max", "smsp__cycles_active.avg", "launch__shared_mem_per_block_dynamic"]
    w = csv.writer(sys.stdout)
    w.writerow(["metric", "unit"] + labels[:len(data)])
    for k in keep:
        if k in hdr:
            i = hdr.index(k)
            w.writerow([k, units[i]] + [d[i] for d in data])
    w.writerow(["gemm_source_sha16", "", gemm_source_sha()] + [""] * (len(data) - 1))
    return 0


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        return dict(hbm_gbs=float(d["hbm_gbs"]), bf16_tflops=float(d["bf16_tflops"]),
                    bf16_tflops_sustained=float(d.get("bf16_tflops_sustained", d["bf16_tflops"])),
                    source="measured (MEASURED_PEAKS.json)")
    return dict(hbm_gbs=6650.0, bf16_tflops=1590.0, bf16_tflops_sustained=1400.0,
                source="fallback (B200_PROFILING.md)")


# ------------------------------------------------------------------ arenas ---
class Arena:
    """One contiguous buffer carved into 256-byte aligned tensors: host (pinned) and device
    mirrors share offsets, so a whole group's inputs move with ONE cudaMemcpyAsync."""

    def __init__(self):
        self.items = []      # (name, offset, host ndarray or None, shape, numpy dtype)
        self.size = 0

    def _push(self, name, a, shape, dtype):
        off = self.size
        self.items.append((name, off, a, tuple(shape), np.dtype(dtype)))
        self.size = (off + int(np.prod(shape)) * np.dtype(dtype).itemsize + 255) & ~255
        return len(self.items) - 1

    def add(self, name, a):
        a = np.ascontiguousarray(a)
        return self._push(name, a, a.shape, a.dtype)

    def reserve(self, name, shape, dt):
        """space only (outputs / intermediates): no host data."""
        return self._push(name, None, shape, np.uint16 if dt == BF16 else np.float32)

    def materialise(self, device, pinned_host):
        import torch
        n = max(self.size, 256)
        self.dev = torch.empty(n, dtype=torch.uint8, device=device)
        self.host = torch.empty(n, dtype=torch.uint8)
        if pinned_host:
            self.host = self.host.pin_memory()
        hv = self.host.numpy()
        for _, off, a, _, _ in self.items:
            if a is not None:
                hv[off:off + a.nbytes] = a.reshape(-1).view(np.uint8)
        if any(a is not None for _, _, a, _, _ in self.items):
            self.dev.copy_(self.host)
        if not pinned_host:
            self.host = None
        return self

    def _span(self, idx):
        _, off, _, shape, dtype = self.items[idx]
        return off, int(np.prod(shape)) * dtype.itemsize, shape, dtype

    def tensor(self, idx):
        """device tensor view of item idx (bf16 or fp32, original shape)."""
        import torch
        off, n, shape, dtype = self._span(idx)
        t = self.dev[off:off + n].view(torch.bfloat16 if dtype == np.uint16 else torch.float32)
        return t.view(*shape)

    def host_array(self, idx):
        off, n, shape, dtype = self._span(idx)
        return self.host.numpy()[off:off + n].view(dtype).reshape(shape)


class Group:
    """One fused op group: a plan (one launch) + what it reads/writes."""

    def __init__(self, name, kind, plan, arena_in, arena_out, bound):
        self.name, self.kind, self.plan, self.ain, self.aout, self.bound = name, kind, plan, arena_in, arena_out, bound
        self.info = plan.info()


class Step:
    """All groups of one step, device-resident, built from the seeded generators."""

    def __init__(self, device="cuda:0", sizes=None, pinned_host=True, configs=("c1", "c2", "c3", "c4")):
        import torch
        import paper_2607_02945_b200 as ob
        self.ob, self.torch, self.device = ob, torch, device
        self.sizes = dict(FULL if sizes is None else sizes)
        self.pinned = pinned_host
        self.groups = []
        dev_index = torch.device(device).index or 0
        self.dev_index = dev_index
        for c in configs:
            getattr(self, "_build_" + c)()

    # ---- C1: batched LayerNorm
    def _build_c1(self):
        ob, s = self.ob, self.sizes
        cfg = wl.config1(rows=s["c1_rows"], n=s["c1_n"])
        ain, aout = Arena(), Arena()
        idx = []
        for m in cfg["members"]:
            idx.append((ain.add("x", m["x"]), ain.add("gamma", m["gamma"]), ain.add("beta", m["beta"]),
                        aout.reserve("y", m["x"].shape, BF16)))
        ain.materialise(self.device, self.pinned), aout.materialise(self.device, self.pinned)
        descs = [ob.layernorm_member(ain.tensor(ix), aout.tensor(iy), ain.tensor(ig), ain.tensor(ib), m["eps"])
                 for (ix, ig, ib, iy), m in zip(idx, cfg["members"])]
        plan = ob.opt_layernorm_plan_create(descs, BF16, BF16, self.dev_index)
        g = Group("C1_batched_layernorm", "layernorm", plan, ain, aout, "hbm")
        g.cfg, g.idx = cfg, idx
        self.groups.append(g)

    # ---- C2: grouped Linear + bias + ReLU, concat output (a2)
    def _build_c2(self):
        ob, s = self.ob, self.sizes
        cfg = wl.config2(M=s["c2_M"], n=s["c2_n"])
        ain, aout = Arena(), Arena()
        idx = [(ain.add("x", m["x"]), ain.add("w", m["w"]), ain.add("b", m["b"])) for m in cfg["members"]]
        iy = aout.reserve("ycat", (cfg["M"], cfg["concat_width"]), BF16)
        ain.materialise(self.device, self.pinned), aout.materialise(self.device, self.pinned)
        ycat = aout.tensor(iy)
        descs = [ob.linear_member(ain.tensor(ix), ain.tensor(iw), ain.tensor(ib),
                                  ycat[:, m["col_off"]:m["col_off"] + m["N"]], m["act"])
                 for (ix, iw, ib), m in zip(idx, cfg["members"])]
        plan = ob.opt_linear_plan_create(descs, BF16, self.dev_index)
        g = Group("C2_grouped_linear_tower", "linear", plan, ain, aout, "tensor")
        g.cfg, g.idx, g.iy = cfg, idx, iy
        self.groups.append(g)

    # ---- C3: split -> pointwise -> cat as one gather/scatter (a4, a5)
    def _build_c3(self):
        ob, s = self.ob, self.sizes
        cfg = wl.config3(rows=s["c3_rows"], width=s["c3_width"], nchunks=s["c3_chunks"])
        ain, aout = Arena(), Arena()
        ix = ain.add("x", cfg["x"])
        iy = aout.reserve("out", cfg["x"].shape, BF16)
        ain.materialise(self.device, self.pinned), aout.materialise(self.device, self.pinned)
        chunks = ob.split_cat_chunks(ain.tensor(ix), aout.tensor(iy), cfg["widths"], cfg["ops"], cfg["perm"])
        plan = ob.opt_pointwise_plan_create(chunks, BF16, self.dev_index)
        g = Group("C3_split_pointwise_cat", "pointwise", plan, ain, aout, "hbm")
        g.cfg, g.ix, g.iy = cfg, ix, iy
        self.groups.append(g)

    # ---- C4: LN group -> GEMM group (+ReLU) -> GEMM group, concat (a6)
    def _build_c4(self):
        ob, s = self.ob, self.sizes
        cfg = wl.config4(B=s["c4_B"], n=s["c4_n"])
        tw = cfg["towers"]
        ain, amid, aout = Arena(), Arena(), Arena()
        idx = []
        for t in tw:
            idx.append(dict(x=ain.add("x", t["x"]), gamma=ain.add("gamma", t["gamma"]), beta=ain.add("beta", t["beta"]),
                            w1=ain.add("w1", t["w1"]), b1=ain.add("b1", t["b1"]), w2=ain.add("w2", t["w2"]),
                            b2=ain.add("b2", t["b2"]),
                            xn=amid.reserve("xn", t["x"].shape, BF16), h=amid.reserve("h", (t["B"], t["H"]), BF16)))
        iy = aout.reserve("out", (cfg["B"], cfg["concat_width"]), BF16)
        ain.materialise(self.device, self.pinned)
        amid.materialise(self.device, False)
        aout.materialise(self.device, self.pinned)
        out = aout.tensor(iy)
        T = ain.tensor
        ln = [ob.layernorm_member(T(i["x"]), amid.tensor(i["xn"]), T(i["gamma"]), T(i["beta"]), t["eps"])
              for i, t in zip(idx, tw)]
        l1 = [ob.linear_member(amid.tensor(i["xn"]), T(i["w1"]), T(i["b1"]), amid.tensor(i["h"]), ACT_RELU)
              for i in idx]
        l2 = [ob.linear_member(amid.tensor(i["h"]), T(i["w2"]), T(i["b2"]), out[:, k * t["out"]:(k + 1) * t["out"]],
                               ACT_NONE) for k, (i, t) in enumerate(zip(idx, tw))]
        empty = Arena().materialise(self.device, self.pinned)
        g1 = Group("C4a_batched_layernorm", "layernorm", ob.opt_layernorm_plan_create(ln, BF16, BF16, self.dev_index),
                   ain, empty, "hbm")
        g2 = Group("C4b_grouped_linear_relu", "linear", ob.opt_linear_plan_create(l1, BF16, self.dev_index),
                   empty, empty, "hbm")
        g3 = Group("C4c_grouped_linear_concat", "linear", ob.opt_linear_plan_create(l2, BF16, self.dev_index),
                   empty, aout, "hbm")
        for g in (g1, g2, g3):
            g.cfg, g.idx, g.amid, g.iy = cfg, idx, amid, iy
        self.groups += [g1, g2, g3]

    # ---- launching
    def launch_all(self, stream=None):
        for g in self.groups:
            g.plan.launch(stream)

    def launch_all_host(self, stream=None, streams=None):
        """e2e: per group, H2D of every input arena, the one kernel, D2H of every output arena --
        all through opt_plan_launch_host (the C ABI call for HOST buffers).  `streams`: one CUDA stream per
        config (C1, C2, C3, C4) -- the configs are independent, so a caller can let their PCIe copies overlap
        (H2D and D2H are separate DMA engines); C4's three dependent groups stay on one stream."""
        ob = self.ob
        for g in self.groups:
            copies = []
            if g.ain.size:
                copies.append(ob.opt_host_copy(g.ain.host.data_ptr(), g.ain.dev.data_ptr(), g.ain.size, 1))
            if g.aout.size:
                copies.append(ob.opt_host_copy(g.aout.host.data_ptr(), g.aout.dev.data_ptr(), g.aout.size, 0))
            s = stream
            if streams is not None:
                s = streams[g.name[:2]].cuda_stream
            g.plan.launch_host(copies, s)

    def h2d_bytes(self):
        return sum(g.ain.size for g in self.groups)

    def d2h_bytes(self):
        return sum(g.aout.size for g in self.groups)


# ------------------------------------------- one-launch-per-op baseline ------
class Unfused:
    """The same groups executed the way the unfused graph runs them: ONE launch per op, through
    single-member plans of the same library (SURVEY.md 8(d) "Baseline"): Linear and its activation are two
    launches, split->f->cat is one launch per chunk plus the cat copy.  Same inputs, same outputs."""

    def __init__(self, step):
        ob, torch = step.ob, step.torch
        self.seq = {}
        self.keep = []
        dev = step.dev_index
        PW_RELU, PW_COPY = 1, 0
        for g in step.groups:
            plans = []
            if g.name.startswith("C1"):
                for (ix, ig, ib, iy), m in zip(g.idx, g.cfg["members"]):
                    d = ob.layernorm_member(g.ain.tensor(ix), g.aout.tensor(iy), g.ain.tensor(ig), g.ain.tensor(ib), m["eps"])
                    plans.append(ob.opt_layernorm_plan_create([d], BF16, BF16, dev))
            elif g.name.startswith("C2"):
                ycat = g.aout.tensor(g.iy)
                for (ix, iw, ib), m in zip(g.idx, g.cfg["members"]):
                    y = ycat[:, m["col_off"]:m["col_off"] + m["N"]]
                    plans.append(ob.opt_linear_plan_create(
                        [ob.linear_member(g.ain.tensor(ix), g.ain.tensor(iw), g.ain.tensor(ib), y, ACT_NONE)], BF16, dev))
                    plans.append(ob.opt_pointwise_plan_create([ob.chunk(y, y, PW_RELU)], BF16, dev))
            elif g.name.startswith("C3"):
                x, out = g.ain.tensor(g.ix), g.aout.tensor(g.iy)
                cfg = g.cfg
                starts = np.concatenate(([0], np.cumsum(cfg["widths"])))
                tmp, cat, d = [], [], 0
                for p in cfg["perm"]:
                    w = cfg["widths"][p]
                    t = torch.empty((x.shape[0], w), dtype=x.dtype, device=x.device)
                    tmp.append(t)
                    plans.append(ob.opt_pointwise_plan_create([ob.chunk(x[:, starts[p]:starts[p] + w], t, cfg["ops"][p])], BF16, dev))
                    cat.append(ob.chunk(t, out[:, d:d + w], PW_COPY))
                    d += w
                plans.append(ob.opt_pointwise_plan_create(cat, BF16, dev))
                self.keep.append(tmp)
            elif g.name.startswith("C4a"):
                T, A = g.ain.tensor, g.amid.tensor
                out = g.aout if g.aout.size else None
                tw = g.cfg["towers"]
                final = step.groups[-1].aout.tensor(g.iy)
                outs, cat = [], []
                for k, (i, t) in enumerate(zip(g.idx, tw)):
                    plans.append(ob.opt_layernorm_plan_create(
                        [ob.layernorm_member(T(i["x"]), A(i["xn"]), T(i["gamma"]), T(i["beta"]), t["eps"])], BF16, BF16, dev))
                for k, (i, t) in enumerate(zip(g.idx, tw)):
                    plans.append(ob.opt_linear_plan_create([ob.linear_member(A(i["xn"]), T(i["w1"]), T(i["b1"]), A(i["h"]), ACT_NONE)], BF16, dev))
                    plans.append(ob.opt_pointwise_plan_create([ob.chunk(A(i["h"]), A(i["h"]), PW_RELU)], BF16, dev))
                for k, (i, t) in enumerate(zip(g.idx, tw)):
                    o = torch.empty((t["B"], t["out"]), dtype=final.dtype, device=final.device)
                    outs.append(o)
                    plans.append(ob.opt_linear_plan_create([ob.linear_member(A(i["h"]), T(i["w2"]), T(i["b2"]), o, ACT_NONE)], BF16, dev))
                    cat.append(ob.chunk(o, final[:, k * t["out"]:(k + 1) * t["out"]], PW_COPY))
                plans.append(ob.opt_pointwise_plan_create(cat, BF16, dev))
                self.keep.append(outs)
                self.seq["C4_recsys_block"] = plans
                continue
            else:
                continue
            self.seq[g.name] = plans

    def time(self, torch, reps=3):
        """-> {group: dict(launches, eager_us, graph_us)}: eager = launches issued one by one from the host
        (what an unfused graph pays); graph = the same sequence replayed as one CUDA graph (GPU-side cost only)."""
        res = {}
        st = torch.cuda.current_stream()
        for name, plans in self.seq.items():
            for p in plans:
                p.launch()
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(st)
            for _ in range(reps):
                for p in plans:
                    p.launch()
            e1.record(st)
            torch.cuda.synchronize()
            eager = e0.elapsed_time(e1) * 1e3 / reps
            graph_us = None
            try:
                gr = torch.cuda.CUDAGraph()
                cs = torch.cuda.Stream()
                cs.wait_stream(st)
                with torch.cuda.graph(gr, stream=cs):
                    for p in plans:
                        p.launch(cs.cuda_stream)
                gr.replay()
                torch.cuda.synchronize()
                e0.record(st)
                for _ in range(reps):
                    gr.replay()
                e1.record(st)
                torch.cuda.synchronize()
                graph_us = e0.elapsed_time(e1) * 1e3 / reps
            except Exception as e:  # noqa: BLE001
                graph_us = None
                self.graph_error = repr(e)
            res[name] = dict(launches=len(plans), eager_us=round(eager, 1), graph_us=None if graph_us is None else round(graph_us, 1))
        return res



# ------------------------------------------------------------- clock watch ---
class ClockWatch(threading.Thread):
    """Samples SM clock, power and throttle reasons through NVML while the timed regions run."""

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.stop_flag, self.samples = index, threading.Event(), []
        self.ok = False
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            # NVML enumerates physical devices; honour CUDA_VISIBLE_DEVICES when it is a plain index list
            vis = os.environ.get("CUDA_VISIBLE_DEVICES")
            phys = index
            if vis:
                try:
                    phys = int(vis.split(",")[index])
                except ValueError:
                    phys = index
            self.h = pynvml.nvmlDeviceGetHandleByIndex(phys)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
            self.ok = True
        except Exception as e:  # noqa: BLE001
            self.err = repr(e)

    def run(self):
        if not self.ok:
            return
        nv = self.nv
        while not self.stop_flag.is_set():
            try:
                mhz = nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)
                reasons = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                util = nv.nvmlDeviceGetUtilizationRates(self.h).gpu
                try:
                    mw = nv.nvmlDeviceGetPowerUsage(self.h)
                except Exception:  # noqa: BLE001
                    mw = None
                self.samples.append((mhz, reasons, util, mw))
            except Exception:  # noqa: BLE001
                pass
            time.sleep(0.01)

    def summary(self):
        if not self.ok or not self.samples:
            return dict(sm_mhz=None, sm_max_mhz=getattr(self, "max_mhz", None), reasons=["unavailable"])
        nv = self.nv
        mhz = sorted(s[0] for s in self.samples)
        bits = 0
        for s in self.samples:
            bits |= s[1]
        names = [("hw_slowdown", nv.nvmlClocksEventReasonHwSlowdown),
                 ("hw_thermal_slowdown", nv.nvmlClocksEventReasonHwThermalSlowdown),
                 ("sw_thermal_slowdown", nv.nvmlClocksEventReasonSwThermalSlowdown),
                 ("sw_power_cap", nv.nvmlClocksEventReasonSwPowerCap),
                 ("hw_power_brake", nv.nvmlClocksEventReasonHwPowerBrakeSlowdown)]
        out = dict(sm_mhz=mhz[len(mhz) // 2], sm_max_mhz=self.max_mhz, samples=len(mhz),
                   reasons=[n for n, b in names if bits & b])
        watts = sorted(s[3] / 1000.0 for s in self.samples if s[3] is not None)
        if watts:
            out["power_w"] = round(watts[len(watts) // 2], 0)
        return out


# ------------------------------------------------------------- CPU oracle ----
def oracle_step(rows, cfgs=None):
    """The oracle, as it stands, over `rows` rows per group of the step's workload (all members, all columns):
    rows = dict(c1_rows, c2_M, c3_rows, c4_B).  cfgs: already generated full-size configs to slice rows from
    (else generated here).  Returns the seconds spent per group [C1, C2, C3, C4]."""
    import oracle
    from oracle import graphs

    def head(a, r):
        return np.ascontiguousarray(a[:r])
    if cfgs is None:
        c1, c2 = wl.config1(rows=rows["c1_rows"]), wl.config2(M=rows["c2_M"])
        c3, c4 = wl.config3(rows=rows["c3_rows"]), wl.config4(B=rows["c4_B"])
    else:   # the first `rows` rows of the full-size tensors (the generators draw row-major: the same values)
        c1 = dict(members=[dict(m, x=head(m["x"], rows["c1_rows"])) for m in cfgs["c1"]["members"]])
        c2 = dict(members=[dict(m, x=head(m["x"], rows["c2_M"])) for m in cfgs["c2"]["members"]])
        c3 = dict(cfgs["c3"], x=head(cfgs["c3"]["x"], rows["c3_rows"]))
        c4 = dict(towers=[dict(t, x=head(t["x"], rows["c4_B"])) for t in cfgs["c4"]["towers"]])
    parts = []
    t = time.perf_counter(); graphs.layernorm_group(c1["members"], BF16); parts.append(time.perf_counter() - t)
    t = time.perf_counter(); graphs.linear_group_concat(c2["members"], BF16); parts.append(time.perf_counter() - t)
    t = time.perf_counter(); graphs.split_pointwise_cat(c3["x"], c3["widths"], c3["ops"], c3["perm"], BF16); parts.append(time.perf_counter() - t)
    t = time.perf_counter()
    outs = [graphs.recsys_tower(tw)["out"] for tw in c4["towers"]]
    oracle.cat(outs)
    parts.append(time.perf_counter() - t)
    return parts


FULL_ROWS = dict(c1_rows=FULL["c1_rows"], c2_M=FULL["c2_M"], c3_rows=FULL["c3_rows"], c4_B=FULL["c4_B"])


def oracle_sample_step(frac=1.0):
    """--impl reference: the oracle on a bounded ROW sample; returns (extrapolated microseconds per full step,
    seconds actually spent, description, cores)."""
    import oracle
    base = dict(c1_rows=2048, c2_M=256, c3_rows=2048, c4_B=128)
    rows = {k: max(8, int(v * frac) // 8 * 8) for k, v in base.items()}
    rows["c1_rows"] = min(rows["c1_rows"], FULL["c1_rows"])
    cores = oracle.max_threads()
    parts = oracle_step(rows)
    scale = [FULL_ROWS[k] / rows[k] for k in ("c1_rows", "c2_M", "c3_rows", "c4_B")]
    spent = sum(parts)
    full_us = sum(p * f for p, f in zip(parts, scale)) * 1e6
    desc = ("rows sampled per group: C1 %d/%d, C2 %d/%d, C3 %d/%d, C4 %d/%d (all members, all columns); "
            "time scaled by rows_full/rows_sampled per group" %
            (rows["c1_rows"], FULL["c1_rows"], rows["c2_M"], FULL["c2_M"], rows["c3_rows"], FULL["c3_rows"],
             rows["c4_B"], FULL["c4_B"]))
    return full_us, spent, desc, cores


def oracle_full_step(cfgs, small=False):
    """cpu_baseline of the product arm (SURVEY 8(d) "CPU oracle timing"): the oracle ONCE over ALL rows of every
    group on all host cores -- measured, not extrapolated -- plus a 1-thread figure on a stated sub-sample."""
    import oracle
    cores = oracle.max_threads()
    rows = dict(FULL_ROWS) if not small else dict(c1_rows=SMALL["c1_rows"], c2_M=SMALL["c2_M"], c3_rows=SMALL["c3_rows"], c4_B=SMALL["c4_B"])
    parts = oracle_step(rows, cfgs)
    sub = {k: max(8, v // 64) for k, v in rows.items()}            # 1 thread: 1/64 of the rows of every group
    oracle.set_threads(1)
    try:
        p1 = oracle_step(sub, cfgs)
    finally:
        oracle.set_threads(cores)
    t1_full_us = sum(p * rows[k] / sub[k] for p, k in zip(p1, ("c1_rows", "c2_M", "c3_rows", "c4_B"))) * 1e6
    return dict(value=round(sum(parts) * 1e6, 1), unit="us", cores=cores, kind="oracle", extrapolated=False,
                sample="ALL rows of every group, once: C1 %d, C2 %d, C3 %d, C4 %d rows (all members, all columns)" %
                       (rows["c1_rows"], rows["c2_M"], rows["c3_rows"], rows["c4_B"]),
                cpu_seconds=round(sum(parts), 2), seconds_per_group=dict(zip(("C1", "C2", "C3", "C4"), [round(p, 2) for p in parts])),
                threads_1=dict(value=round(t1_full_us, 1), unit="us", extrapolated=True, cpu_seconds=round(sum(p1), 2),
                               sample="1 thread on 1/64 of the rows of every group (C1 %d, C2 %d, C3 %d, C4 %d), scaled by 64" %
                                      (sub["c1_rows"], sub["c2_M"], sub["c3_rows"], sub["c4_B"])))


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    K, W = args.steps, args.warmup
    frac = min(1.0, (100.0 / max(1, K + W)) / 8.0)          # whole run ~100 s of CPU work
    if args.ref_frac:
        frac = args.ref_frac
    vals, spent_all, desc, cores = [], 0.0, "", 0
    for i in range(W + K):
        us, spent, desc, cores = oracle_sample_step(frac)
        if i >= W:
            vals.append(us)
            spent_all += spent
    v = float(np.mean(vals))
    line = dict(metric="fused_op_group_step_latency", value=v, unit="us", n_gpus=args.gpus, steps=K, warmup=W,
                ms_per_step=v / 1e3, higher_is_better=False, scaling="weak", vs_baseline=None, dtype="f64",
                data="synthetic", impl="reference",
                config=dict(workload=WORKLOAD_NAME, l2="n/a (CPU)"),
                cpu_baseline=dict(value=v, unit="us", cores=cores, kind="oracle", sample=desc, extrapolated=True,
                                  measured_seconds_per_step=spent_all / max(1, K), measured_seconds_total=spent_all,
                                  note="each step times the oracle on the row sample; value = that time scaled by "
                                       "rows_full / rows_sampled per group (the full-size oracle pass, ~40 s, is timed once "
                                       "in the product arm's cpu_baseline)"),
                e2e=dict(value=v, unit="us", h2d_bytes_per_step=0, d2h_bytes_per_step=0), gpu_launches=0)
    print(json.dumps(line))
    return 0


WORKLOAD_NAME = ("whole hot path = fused groups of BASELINE.json configs[1..4] back to back: C1 batched LN x64, "
                 "C2 grouped Linear+ReLU x128 (M=4096, concat), C3 split-pointwise-cat 8192x8192/256 chunks, "
                 "C4 recsys block x512 (LN -> Linear+ReLU -> Linear, concat [8192,32768]); 6 launches/step")


def max_over_ranks(values, world, device):
    """Timing rule: a multi-rank number is the MAX over ranks (replicas only).
    One all_reduce(MAX) on whatever backend the process group has (nccl on GPUs, gloo in the CPU test)."""
    if world <= 1:
        return [float(v) for v in values]
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(v) for v in values], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(v) for v in t.tolist()]


def aggregate_steps_per_s(us_step, world):
    """whole-job throughput of `world` independent replicas whose slowest rank needs us_step per step."""
    return world / (us_step * 1e-6)


# ------------------------------------------------------- side workloads ------
def run_side(args):
    """Small stand-alone workloads for ncu captures of the section-8(f) items (profiles/r01_profiles.md section 4):
      --side linear2   C4's two GEMM groups as one chained-Linear launch (opt_linear2), 3 launches
      --side ln_linear2  the whole C4 block (LayerNorm folded into the chain, opt_ln_linear2) as one launch
      --side skinny    the paper's four skinny aten.mm as one group (streaming row kernel)
      --side fp8       configs[4]'s saved LayerNorm outputs -> FP8 E4M3 and back (one launch each)
      --side bias_grad the 512 bias gradients of configs[4]'s Linear+ReLU group (column sums of [8192, H]), one launch
      --side fp8_fused configs[4]'s LayerNorm and Linear+ReLU groups writing bf16 AND the FP8 copy in one launch vs two launches
      --side backward  configs[2] dgrad / wgrad / fused mask + bias gradient, configs[4] LayerNorm backward, one launch each
      --side gemm_trace  wait-cycle counters of the grouped GEMM's warp roles (trace build of the library)
      --side linear2_trace  the same for the chained kernel (opt_linear2 / opt_ln_linear2 on configs[4]'s towers)
      --side power       every group launched back to back for 1.5 s: time, board power, SM clock (what the power cap does)
      --side lhs       batch_linear_lhs: 8 members (N=64) on ONE input X [262144, 512]; also timed with
                       opt_linear_options.no_lhs_order (plain member-major schedule)
    Prints one JSON line; not the bench metric."""
    import torch
    from ctypes import c_void_p as C_void_p
    import paper_2607_02945_b200 as ob
    torch.cuda.set_device(0)
    stream = torch.cuda.current_stream()

    def timed(fn, n=5):
        flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device="cuda")
        ts = []
        for _ in range(n):
            flush.fill_(1)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream); fn(); e1.record(stream)
            torch.cuda.synchronize()
            ts.append(e0.elapsed_time(e1) * 1e3)
        return float(np.mean(ts))

    if args.side == "linear2":
        step = Step("cuda:0", FULL, pinned_host=False, configs=("c4",))
        ga, gb, gc = step.groups
        T, A = ga.ain.tensor, ga.amid.tensor
        out2 = torch.empty_like(gc.aout.tensor(ga.iy))
        descs = [ob.linear2_member(A(i["xn"]), T(i["w1"]), T(i["b1"]), T(i["w2"]), T(i["b2"]),
                                   out2[:, k * t["out"]:(k + 1) * t["out"]], ACT_RELU, ACT_NONE)
                 for k, (i, t) in enumerate(zip(ga.idx, ga.cfg["towers"]))]
        plan = ob.opt_linear2_plan_create(descs, BF16, 0)
        ga.plan.launch()
        torch.cuda.synchronize()
        print(json.dumps(dict(side="linear2", us=round(timed(plan.launch, 3), 1), **plan.info())))
    elif args.side == "ln_linear2":
        step = Step("cuda:0", FULL, pinned_host=False, configs=("c4",))
        ga = step.groups[0]
        T = ga.ain.tensor
        out3 = torch.empty_like(step.groups[2].aout.tensor(ga.iy))
        plan = ob.opt_ln_linear2_plan_create(
            [ob.ln_linear2_member(T(i["x"]), T(i["gamma"]), T(i["beta"]), t["eps"], T(i["w1"]), T(i["b1"]), T(i["w2"]), T(i["b2"]),
                                  out3[:, k * t["out"]:(k + 1) * t["out"]], ACT_RELU, ACT_NONE)
             for k, (i, t) in enumerate(zip(ga.idx, ga.cfg["towers"]))], BF16, 0)
        plan.launch()
        torch.cuda.synchronize()
        print(json.dumps(dict(side="ln_linear2", us=round(timed(plan.launch, 3), 1), **plan.info())))
    elif args.side == "backward":
        # backward groups at full size, one launch each (for ncu): configs[2] dgrad, wgrad, fused ReLU-mask + bias gradient;
        # configs[4] LayerNorm-group backward
        step = Step("cuda:0", FULL, pinned_host=False, configs=("c2",))
        g2 = step.groups[0]
        g2.plan.launch()
        ycat = g2.aout.tensor(g2.iy)
        dy_cat = torch.empty_like(ycat).normal_(0.0, 1.0)
        dg, wg, bg, keep = [], [], [], []
        for (ix, iw, ib), m in zip(g2.idx, g2.cfg["members"]):
            x, w = g2.ain.tensor(ix), g2.ain.tensor(iw)
            sl = slice(m["col_off"], m["col_off"] + m["N"])
            dx, dw, db = torch.empty_like(x), torch.empty_like(w), torch.empty(m["N"], dtype=torch.float32, device="cuda")
            keep.append((dx, dw, db))
            dg.append(ob.linear_member(dy_cat[:, sl], w, None, dx, ACT_NONE, ob.OPT_LAYOUT_W_TRANSPOSED))
            wg.append(ob.linear_member(dy_cat[:, sl], x, None, dw, ACT_NONE, ob.OPT_LAYOUT_X_TRANSPOSED | ob.OPT_LAYOUT_W_TRANSPOSED))
            bg.append(ob.bias_grad_member(dy_cat[:, sl], db, ycat[:, sl], dy_cat[:, sl], ob.OPT_ACT_RELU))
        pb = ob.opt_bias_grad_plan_create(bg, BF16, ob.OPT_F32, 0)
        pd, pw = ob.opt_linear_plan_create(dg, BF16, 0), ob.opt_linear_plan_create(wg, BF16, 0)
        for p_ in (pb, pd, pw):
            p_.launch()
        torch.cuda.synchronize()
        res = dict(side="backward", c2_mask_bias_grad_us=round(timed(pb.launch, 3), 1), c2_dgrad_us=round(timed(pd.launch, 3), 1),
                   c2_wgrad_us=round(timed(pw.launch, 3), 1), c2_dgrad_flops=pd.info()["flops"], c2_mask_bias_grad_bytes=pb.info()["bytes"])
        del step, g2, keep, dy_cat, pb, pd, pw
        cfg4 = wl.config4()
        lb, keep = [], []
        for t in cfg4["towers"]:
            x = torch.from_numpy(t["x"].view(np.int16)).cuda().view(torch.bfloat16)
            gam = torch.from_numpy(t["gamma"].view(np.int16)).cuda().view(torch.bfloat16)
            dyl = torch.empty_like(x).normal_(0.0, 1.0)
            dxl, dgl, dbl = torch.empty_like(x), torch.empty_like(gam), torch.empty_like(gam)
            keep.append((x, gam, dyl, dxl, dgl, dbl))
            lb.append(ob.layernorm_bwd_member(x, dyl, gam, dxl, dgl, dbl, 1e-5))
        pl = ob.opt_layernorm_bwd_plan_create(lb, BF16, BF16, 0)
        pl.launch()
        torch.cuda.synchronize()
        res.update(c4_layernorm_bwd_us=round(timed(pl.launch, 3), 1), c4_layernorm_bwd_bytes=pl.info()["bytes"])
        print(json.dumps(res))
    elif args.side == "fp8_fused":
        # activation quantisation fused into the producer: configs[4]'s LayerNorm group writing its bf16
        # output AND the FP8 copy in one launch, next to LayerNorm + OPT_PW_QUANT_E4M3 (two launches); same for C4b's GEMM
        step = Step("cuda:0", FULL, pinned_host=False, configs=("c4",))
        ga, gb, gc = step.groups
        T, A = ga.ain.tensor, ga.amid.tensor
        q8 = [torch.empty(A(i["xn"]).shape, dtype=torch.uint8, device="cuda") for i in ga.idx]
        pf = ob.opt_layernorm_plan_create([ob.layernorm_member(T(i["x"]), A(i["xn"]), T(i["gamma"]), T(i["beta"]), t["eps"], q, 16.0)
                                           for i, t, q in zip(ga.idx, ga.cfg["towers"], q8)], BF16, BF16, 0)
        pq = ob.opt_pointwise_plan_create([ob.chunk(A(i["xn"]), q, ob.OPT_PW_QUANT_E4M3, None, [16.0]) for i, q in zip(ga.idx, q8)], BF16, 0)
        h8 = [torch.empty(A(i["h"]).shape, dtype=torch.uint8, device="cuda") for i in ga.idx]
        pg = ob.opt_linear_plan_create([ob.linear_member(A(i["xn"]), T(i["w1"]), T(i["b1"]), A(i["h"]), ACT_RELU, 0, q, 8.0)
                                        for i, q in zip(ga.idx, h8)], BF16, 0)
        ph = ob.opt_pointwise_plan_create([ob.chunk(A(i["h"]), q, ob.OPT_PW_QUANT_E4M3, None, [8.0]) for i, q in zip(ga.idx, h8)], BF16, 0)
        for p_ in (ga.plan, pf, pq, gb.plan, pg, ph):
            p_.launch()
        torch.cuda.synchronize()
        print(json.dumps(dict(side="fp8_fused", ln_us=round(timed(ga.plan.launch, 3), 1), ln_with_fp8_copy_us=round(timed(pf.launch, 3), 1),
                              quant_launch_us=round(timed(pq.launch, 3), 1), ln_bytes=ga.plan.info()["bytes"], ln_with_fp8_bytes=pf.info()["bytes"],
                              gemm_us=round(timed(gb.plan.launch, 3), 1), gemm_with_fp8_copy_us=round(timed(pg.launch, 3), 1),
                              gemm_quant_launch_us=round(timed(ph.launch, 3), 1), gemm_bytes=gb.plan.info()["bytes"], gemm_with_fp8_bytes=pg.info()["bytes"])))
    elif args.side == "skinny":
        shapes = [(18583840, 8, 8), (25247936, 4, 2), (22502112, 8, 8), (17980096, 4, 2)]       # PAPER.md:477, (M, K, N)
        ten = [(torch.randn(M, K, device="cuda", dtype=torch.bfloat16), torch.randn(N, K, device="cuda", dtype=torch.bfloat16),
                torch.empty(M, N, device="cuda", dtype=torch.bfloat16)) for M, K, N in shapes]
        plan = ob.opt_linear_plan_create([ob.linear_member(x, w, None, y, ACT_NONE) for x, w, y in ten], BF16, 0)
        plan.launch()
        torch.cuda.synchronize()
        print(json.dumps(dict(side="skinny", us=round(timed(plan.launch, 3), 1), **plan.info())))
    elif args.side == "bias_grad":
        rng = np.random.default_rng(4)
        hs = [int(h) for h in rng.choice([128, 256, 512], size=512)]                          # configs[4]'s hidden widths
        dz = [torch.randn(8192, h, device="cuda", dtype=torch.bfloat16) for h in hs]
        db = [torch.empty(h, device="cuda", dtype=torch.float32) for h in hs]
        plan = ob.opt_bias_grad_plan_create([ob.bias_grad_member(z, d) for z, d in zip(dz, db)], BF16, ob.OPT_F32, 0)
        plan.launch()
        torch.cuda.synchronize()
        res = dict(side="bias_grad", us=round(timed(plan.launch, 5), 1), **plan.info())
        # the ReLU mask fused in front: dZ = dY where y > 0, written once and summed in the same pass (3 M N elements of
        # traffic) against the two-launch path OPT_PW_RELU_BWD + bias gradient (4 M N)
        ys = [torch.randn(8192, h, device="cuda", dtype=torch.bfloat16).clamp_(min=0) for h in hs]
        outs = [torch.empty_like(z) for z in dz]
        pf = ob.opt_bias_grad_plan_create([ob.bias_grad_member(z, d, y, o) for z, d, y, o in zip(dz, db, ys, outs)], BF16, ob.OPT_F32, 0)
        pm = ob.opt_pointwise_plan_create([ob.chunk(z, o, ob.OPT_PW_RELU_BWD, y) for z, y, o in zip(dz, ys, outs)], BF16, 0)
        pb2 = ob.opt_bias_grad_plan_create([ob.bias_grad_member(o, d) for o, d in zip(outs, db)], BF16, ob.OPT_F32, 0)
        pf.launch(); pm.launch(); pb2.launch()
        torch.cuda.synchronize()
        res.update(fused_mask_us=round(timed(pf.launch, 5), 1), fused_mask_bytes=pf.info()["bytes"],
                   two_launch_us=round(timed(lambda: (pm.launch(), pb2.launch()), 5), 1),
                   two_launch_bytes=pm.info()["bytes"] + pb2.info()["bytes"])
        print(json.dumps(res))
    elif args.side == "gemm_trace":
        # where the grouped GEMM's warp roles wait: the pipeline-trace build of the library (-DOPTB_GEMM_TRACE; a
        # separate .so) adds up clock64() cycles spent blocked per barrier, one record per CTA.  Workloads: configs[2]
        # (with the ring-depth sensitivity) and the batch_linear_lhs side group (8 x N=64 on one X).
        from paper_2607_02945_b200 import binding
        binding.use_trace_library()
        grid = 148
        buf = torch.zeros(grid * 16, dtype=torch.int64, device="cuda")
        assert binding.lib().opt_trace_set_gemm_buffer(C_void_p(buf.data_ptr())) == 0
        flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device="cuda")

        def trace(plan):
            for _ in range(3):
                plan.launch()
            torch.cuda.synchronize()
            us = timed(plan.launch, 5)
            buf.zero_()
            flush.fill_(1)
            plan.launch()
            torch.cuda.synchronize()
            r = buf.cpu().numpy().reshape(grid, 16).astype(np.float64)
            lead, peer = r[0::2], r[1::2]
            pct = lambda a, tot: [round(float(v), 1) for v in np.percentile(100.0 * a / np.maximum(tot, 1), [0, 50, 100])]
            return dict(us=round(us, 1), pairs=int(lead.shape[0]),
                        mma_total_cycles_min_med_max=[int(v) for v in np.percentile(lead[:, 3], [0, 50, 100])],
                        mma_wait_full_pct=pct(lead[:, 5], lead[:, 3]), mma_wait_tempty_pct=pct(lead[:, 6], lead[:, 3]),
                        mma_wait_queue_pct=pct(lead[:, 4], lead[:, 3]),
                        mma_issue_pct=pct(lead[:, 3] - lead[:, 4] - lead[:, 5] - lead[:, 6], lead[:, 3]),
                        tiles_per_pair_min_med_max=[int(v) for v in np.percentile(lead[:, 7], [0, 50, 100])],
                        tensor_cycles_per_pair_min_med_max=[int(v) for v in np.percentile(lead[:, 8] * 2, [0, 50, 100])],
                        tensor_busy_pct=pct(lead[:, 8] * 2, lead[:, 3]),
                        producer_wait_empty_pct=pct(lead[:, 2], lead[:, 0]), producer_wait_queue_pct=pct(lead[:, 1], lead[:, 0]),
                        peer_producer_wait_empty_pct=pct(peer[:, 2], peer[:, 0]),
                        epilogue_wait_tfull_pct=pct(lead[:, 11], lead[:, 9]), epilogue_wait_store_pct=pct(lead[:, 12], lead[:, 9]),
                        epilogue_wait_queue_pct=pct(lead[:, 10], lead[:, 9]))

        step = Step("cuda:0", FULL, pinned_host=False, configs=("c2",))
        g = step.groups[0]
        c2 = trace(g.plan)
        depth = {}
        for ns in (2, 3, 4, 5):        # ring-depth sensitivity (trace build only): latency-bound or bandwidth-bound?
            o = ob.opt_linear_options(); o.reserved[0] = ns
            ycat = g.aout.tensor(g.iy)
            pd = ob.opt_linear_plan_create_ex([ob.linear_member(g.ain.tensor(ix), g.ain.tensor(iw), g.ain.tensor(ib),
                                                                 ycat[:, m["col_off"]:m["col_off"] + m["N"]], m["act"])
                                               for (ix, iw, ib), m in zip(g.idx, g.cfg["members"])], BF16, 0, o)
            pd.launch(); torch.cuda.synchronize()
            depth[str(ns)] = round(timed(pd.launch, 5), 1)
        c2["us_by_ring_stages"] = depth
        del step, g
        step4 = Step("cuda:0", FULL, pinned_host=False, configs=("c4",))       # the two HBM-bound GEMM groups of configs[4]
        for g4 in step4.groups:
            g4.plan.launch()
        torch.cuda.synchronize()
        c4 = {g4.name: trace(g4.plan) for g4 in step4.groups if g4.kind == "linear"}
        del step4
        M, K, N, n = 262144, 512, 64, 8
        gen = torch.Generator(device="cuda").manual_seed(0)
        x = torch.randn(M, K, device="cuda", generator=gen).to(torch.bfloat16)
        ws = [(torch.randn(N, K, device="cuda", generator=gen) * K ** -0.5).to(torch.bfloat16) for _ in range(n)]
        ycat = torch.empty(M, N * n, device="cuda", dtype=torch.bfloat16)
        lhs = trace(ob.opt_linear_plan_create([ob.linear_member(x, w, None, ycat[:, i * N:(i + 1) * N], ACT_RELU) for i, w in enumerate(ws)], BF16, 0))
        print(json.dumps(dict(side="gemm_trace", configs2=c2, configs4=c4, batch_linear_lhs_8xN64=lhs,
                              note="percentages of the role's own loop time, [min, median, max] over the CTA pairs; tensor cycles = "
                                   "sum over tiles of k-blocks x (BN / 256) x 512 (a 256 x 256 x 64 k-block keeps the pair's tensor "
                                   "pipes busy for 512 cycles)")))
    elif args.side == "linear2_trace":
        # where the chained kernel's warp roles wait (trace build of the library, like gemm_trace): one record of 32
        # counters per CTA, for opt_linear2 and opt_ln_linear2 on configs[4]'s towers
        from paper_2607_02945_b200 import binding
        binding.use_trace_library()
        step = Step("cuda:0", FULL, pinned_host=False, configs=("c4",))
        ga, gb, gc = step.groups
        T, A = ga.ain.tensor, ga.amid.tensor
        out2 = torch.empty_like(gc.aout.tensor(ga.iy))
        ga.plan.launch()
        torch.cuda.synchronize()
        grid = 148
        buf = torch.zeros(grid * 32, dtype=torch.int64, device="cuda")
        assert binding.lib().opt_trace_set_linear2_buffer(C_void_p(buf.data_ptr())) == 0
        flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device="cuda")
        roles = {"producer": (0, dict(queue=1, x_empty=2, w1_empty=3, w2_empty=4)),
                 "mma1": (5, dict(queue=6, acc1_empty=7, x_full=8, w1_full=9)),
                 "mma2": (12, dict(queue=13, acc2_empty=14, w2_full=15, h_full=16)),
                 "epilogue": (17, dict(queue=18, acc1_full=19, h_empty=20, acc2_full=21, store=22, drain_total=23, x_full=24,
                                       seg_tmem_load=25, seg_math=26, seg_hidden_store=27, seg_publish=28))}

        def trace(plan):
            for _ in range(3):
                plan.launch()
            torch.cuda.synchronize()
            us = timed(plan.launch, 5)
            buf.zero_()
            flush.fill_(1)
            plan.launch()
            torch.cuda.synchronize()
            r = buf.cpu().numpy().reshape(grid, 32).astype(np.float64)
            pct = lambda a, tot: [round(float(v), 1) for v in np.percentile(100.0 * a / np.maximum(tot, 1), [0, 50, 100])]
            out = dict(us=round(us, 1))
            for role, (tot, d) in roles.items():
                out[role] = dict(total_cycles_min_med_max=[int(v) for v in np.percentile(r[:, tot], [0, 50, 100])],
                                 **{k + "_pct": pct(r[:, i], r[:, tot]) for k, i in d.items()})
            out["tiles_per_cta_min_med_max"] = [int(v) for v in np.percentile(r[:, 10], [0, 50, 100])]
            out["hidden_chunks_per_cta_min_med_max"] = [int(v) for v in np.percentile(r[:, 29], [0, 50, 100])]
            out["epilogue_cycles_per_chunk"] = {k: round(float(np.median(r[:, i] / np.maximum(r[:, 29], 1))), 1)
                                                for k, i in dict(tmem_load=25, math=26, hidden_store=27, publish=28).items()}
            out["tensor_busy_pct"] = pct(r[:, 11], r[:, 5])
            return out

        towers = list(enumerate(zip(ga.idx, ga.cfg["towers"])))
        p2 = ob.opt_linear2_plan_create([ob.linear2_member(A(i["xn"]), T(i["w1"]), T(i["b1"]), T(i["w2"]), T(i["b2"]),
                                                           out2[:, k * t["out"]:(k + 1) * t["out"]], ACT_RELU, ACT_NONE) for k, (i, t) in towers], BF16, 0)
        res = dict(side="linear2_trace", linear2=trace(p2))
        del p2
        pl = ob.opt_ln_linear2_plan_create([ob.ln_linear2_member(T(i["x"]), T(i["gamma"]), T(i["beta"]), t["eps"], T(i["w1"]), T(i["b1"]), T(i["w2"]),
                                                                 T(i["b2"]), out2[:, k * t["out"]:(k + 1) * t["out"]], ACT_RELU, ACT_NONE)
                                            for k, (i, t) in towers], BF16, 0)
        res["ln_linear2"] = trace(pl)
        res["note"] = ("percentages of the role's own loop time, [min, median, max] over the 148 CTAs; tensor cycles = per hidden chunk "
                       "(chunk width / 2) x K=16 steps of layer 1 + (chunk width / 16) x (N / 2) of layer 2")
        print(json.dumps(res))
    elif args.side == "power":
        # What the power cap does to each group: a group launched back to back for 1.5 s (no L2 flush, no gaps), with SM
        # clock and board power sampled through NVML; next to a device copy and a cuBLAS GEMM as references.  The step's
        # 50-step timed region (about 90 ms) sits between the burst figures (isolated, cold L2) and these sustained ones.
        step = Step("cuda:0", FULL, pinned_host=False)

        def sustained(fn, seconds=1.5, batch=50):
            for _ in range(20):
                fn()
            torch.cuda.synchronize()
            w = ClockWatch(0)
            w.start()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            t0, n = time.time(), 0
            e0.record()
            while time.time() - t0 < seconds:
                for _ in range(batch):
                    fn()
                n += batch
                torch.cuda.synchronize()
            e1.record()
            torch.cuda.synchronize()
            w.stop_flag.set()
            w.join(timeout=2)
            c = w.summary()
            us = e0.elapsed_time(e1) * 1e3 / n
            return dict(us=round(us, 1), power_w=c.get("power_w"), sm_mhz=c.get("sm_mhz"), sm_max_mhz=c.get("sm_max_mhz"),
                        joule_per_launch=None if c.get("power_w") is None else round(c["power_w"] * us * 1e-6, 3))

        res = dict(side="power")
        for g in step.groups:
            res[g.name] = dict(sustained(g.plan.launch), algorithmic_bytes=g.info["bytes"])

        def whole():
            for g in step.groups:
                g.plan.launch()
        res["step"] = sustained(whole, 3.0, 10)
        del step
        a = torch.empty(1500 * 1024 * 1024, dtype=torch.uint8, device="cuda")
        b = torch.empty_like(a)
        res["device_copy_3.1GB"] = dict(sustained(lambda: b.copy_(a)), algorithmic_bytes=2 * a.numel())
        del a, b
        x = torch.randn(8192, 8192, device="cuda", dtype=torch.bfloat16)
        res["cublas_bf16_8192^3"] = dict(sustained(lambda: torch.matmul(x, x)), flops=2 * 8192 ** 3)
        print(json.dumps(res))
    elif args.side == "fp8":
        step = Step("cuda:0", FULL, pinned_host=False, configs=("c4",))
        ga = step.groups[0]
        ga.plan.launch()
        A = ga.amid.tensor
        q8 = [torch.empty(A(i["xn"]).shape, dtype=torch.uint8, device="cuda") for i in ga.idx]
        r16 = [torch.empty_like(A(i["xn"])) for i in ga.idx]
        pq = ob.opt_pointwise_plan_create([ob.chunk(A(i["xn"]), q, ob.OPT_PW_QUANT_E4M3, None, [16.0]) for i, q in zip(ga.idx, q8)], BF16, 0)
        pdq = ob.opt_pointwise_plan_create([ob.chunk(q, r, ob.OPT_PW_DEQUANT_E4M3, None, [1.0 / 16.0]) for q, r in zip(q8, r16)], BF16, 0)
        pq.launch(); pdq.launch()
        torch.cuda.synchronize()
        print(json.dumps(dict(side="fp8", quant_us=round(timed(pq.launch, 3), 1), dequant_us=round(timed(pdq.launch, 3), 1),
                              quant_bytes=pq.info()["bytes"], dequant_bytes=pdq.info()["bytes"])))
    else:
        M, K, N, n = 262144, 512, 64, 8
        g = torch.Generator(device="cuda").manual_seed(0)
        x = torch.randn(M, K, device="cuda", generator=g).to(torch.bfloat16)
        ws = [(torch.randn(N, K, device="cuda", generator=g) * K ** -0.5).to(torch.bfloat16) for _ in range(n)]
        ycat = torch.empty(M, N * n, device="cuda", dtype=torch.bfloat16)
        descs = [ob.linear_member(x, w, None, ycat[:, i * N:(i + 1) * N], ACT_RELU) for i, w in enumerate(ws)]
        plan = ob.opt_linear_plan_create(descs, BF16, 0)
        plain = ob.opt_linear_plan_create_ex(descs, BF16, 0, ob.opt_linear_options(no_lhs_order=1))
        plan.launch(); plain.launch()
        torch.cuda.synchronize()
        print(json.dumps(dict(side="lhs", us=round(timed(plan.launch, 3), 1), us_member_major_order=round(timed(plain.launch, 3), 1),
                              **plan.info())))
    return 0


# -------------------------------------------------------------- product arm --
def run_product(args):
    import torch
    import torch.distributed as dist
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the product path has no CPU fallback")
    torch.cuda.set_device(local)
    device = "cuda:%d" % local
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device(device))
    import paper_2607_02945_b200 as ob

    peaks = load_peaks()
    K, W = args.steps, max(args.warmup, 3)
    t0 = time.time()
    step = Step(device, SMALL if args.small else FULL, pinned_host=True)
    build_s = time.time() - t0
    stream = torch.cuda.current_stream()
    ng = len(step.groups)

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    watch = ClockWatch(local)
    watch.start()

    # ---- (1) device-resident: W warm-ups, then EXACTLY K steps between two events
    for _ in range(W):
        step.launch_all()
    barrier()
    n0 = ob.opt_launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(K):
        step.launch_all()
    e1.record(stream)
    barrier()
    launches = ob.opt_launch_count() - n0
    ms_total = e0.elapsed_time(e1)

    # ---- (2) same K steps again with an event pair around every launch -> per-group durations
    evs = [[(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(ng)]
           for _ in range(K)]
    for k in range(K):
        for gi, g in enumerate(step.groups):
            evs[k][gi][0].record(stream)
            g.plan.launch()
            evs[k][gi][1].record(stream)
    barrier()
    per_group_us = [float(np.mean([evs[k][gi][0].elapsed_time(evs[k][gi][1]) for k in range(K)])) * 1e3
                    for gi in range(ng)]
    per_group_min_us = [float(np.min([evs[k][gi][0].elapsed_time(evs[k][gi][1]) for k in range(K)])) * 1e3
                        for gi in range(ng)]

    # ---- (3) end to end through opt_plan_launch_host: pinned host -> device, kernel, device -> host
    Ke = max(1, min(K, args.e2e_steps))
    for _ in range(2):
        step.launch_all_host()
    barrier()
    f0, f1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    f0.record(stream)
    for _ in range(Ke):
        step.launch_all_host()
    f1.record(stream)
    barrier()
    ms_e2e = f0.elapsed_time(f1)
    # the same, the four independent configs on four streams (copies of one config overlap the others')
    side = {k: torch.cuda.Stream() for k in ("C1", "C2", "C3", "C4")}
    step.launch_all_host(streams=side)
    barrier()
    f2, f3 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    f2.record(stream)
    for st_ in side.values():
        st_.wait_stream(stream)
    for _ in range(Ke):
        step.launch_all_host(streams=side)
    for st_ in side.values():
        stream.wait_stream(st_)
    f3.record(stream)
    barrier()
    ms_e2e_ms = f2.elapsed_time(f3)

    # ---- (4) size-matched plain-copy reference for the HBM-bound groups: a device-to-device copy of the same
    # number of bytes (half read, half written), cold L2, same event protocol.  Small groups cannot reach the
    # large-copy peak whatever the kernel: launch ramp and tail are a fixed ~8 us.
    copy_ref, isolated = {}, {}
    flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device=device)
    for g in step.groups:
        if args.profile:
            continue
        with_copy = g.kind != "linear"
        if with_copy:
            n = g.info["bytes"] // 2
            a = torch.empty(n, dtype=torch.uint8, device=device)
            b = torch.empty(n, dtype=torch.uint8, device=device)
            b.copy_(a)
        ts, tk = [], []
        for _ in range(10):
            if with_copy:
                flush.fill_(1)
                c0, c1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                c0.record(stream); b.copy_(a); c1.record(stream)
                torch.cuda.synchronize()
                ts.append(c0.elapsed_time(c1) * 1e3)
            flush.fill_(1)
            c0, c1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            c0.record(stream); g.plan.launch(); c1.record(stream)
            torch.cuda.synchronize()
            tk.append(c0.elapsed_time(c1) * 1e3)
        isolated[g.name] = float(np.mean(tk))
        if with_copy:
            copy_ref[g.name] = (float(np.mean(ts)), float(np.mean(tk)))
            del a, b
    del flush

    # ---- (5) one-launch-per-op baseline (same library, single-member plans), outside the timed step
    unfused = None
    if not args.no_unfused and not args.profile:
        try:
            unfused = Unfused(step).time(torch)
        except Exception as e:  # noqa: BLE001
            unfused = dict(error=repr(e))

    # ---- (5b) configs[0] (tiny fp32 group, launch-latency bound): latency of the one fused launch next to the
    # eight launches of the unfused graph (4 x Linear + 4 x tanh), 200 back-to-back launches each; no roofline claim
    c0 = None
    if not args.profile:
        try:
            cfg0 = wl.config0()
            t32 = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(device)
            d0 = [(t32(m["x"]), t32(m["w"]), t32(m["b"]), torch.empty((m["M"], m["N"]), dtype=torch.float32, device=device))
                  for m in cfg0["members"]]
            fused = ob.opt_linear_plan_create([ob.linear_member(x, w, b, y, m["act"]) for (x, w, b, y), m in zip(d0, cfg0["members"])], F32, step.dev_index)
            singles = []
            for (x, w, b, y), m in zip(d0, cfg0["members"]):
                singles.append(ob.opt_linear_plan_create([ob.linear_member(x, w, b, y, ACT_NONE)], F32, step.dev_index))
                singles.append(ob.opt_pointwise_plan_create([ob.chunk(y, y, m["act"])], F32, step.dev_index))

            def lat(fn, n=200):
                for _ in range(10):
                    fn()
                torch.cuda.synchronize()
                a, b_ = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record(stream)
                for _ in range(n):
                    fn()
                b_.record(stream)
                torch.cuda.synchronize()
                return a.elapsed_time(b_) * 1e3 / n
            def graph_lat(plans, reps=50):      # the same launches replayed from one CUDA graph: GPU-side latency only
                gr, cs = torch.cuda.CUDAGraph(), torch.cuda.Stream()
                cs.wait_stream(stream)
                with torch.cuda.graph(gr, stream=cs):
                    for _ in range(reps):
                        for p_ in plans:
                            p_.launch(cs.cuda_stream)
                gr.replay()
                torch.cuda.synchronize()
                a, b_ = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record(stream)
                for _ in range(4):
                    gr.replay()
                b_.record(stream)
                torch.cuda.synchronize()
                return a.elapsed_time(b_) * 1e3 / (4 * reps)
            c0 = dict(workload="configs[0]: 4 Linear+bias+tanh members, fp32, M=64", fused_launches=1,
                      fused_us=round(lat(fused.launch), 2), fused_graph_us=round(graph_lat([fused]), 2),
                      unfused_launches=len(singles), unfused_us=round(lat(lambda: [p.launch() for p in singles]), 2),
                      unfused_graph_us=round(graph_lat(singles), 2),
                      note="*_us: launched one by one from the host (Python + ctypes: host-bound); *_graph_us: replayed "
                           "from a CUDA graph")
        except Exception as e:  # noqa: BLE001
            c0 = dict(error=repr(e))

    # ---- (6) SURVEY 8(f) rank 1, side figure (NOT part of the step): C4's two GEMM groups as ONE chained-Linear
    # launch (opt_linear2, hidden tensor on chip) next to the two-launch path, isolated, cold L2, same tensors
    vertical = None
    c4 = [g for g in step.groups if g.name.startswith("C4")]
    if len(c4) == 3 and not args.profile and not args.small:
        try:
            ga, gb, gc = c4
            T, A = ga.ain.tensor, ga.amid.tensor
            ref_out = gc.aout.tensor(ga.iy)
            out2 = torch.empty_like(ref_out)
            descs = [ob.linear2_member(A(i["xn"]), T(i["w1"]), T(i["b1"]), T(i["w2"]), T(i["b2"]),
                                       out2[:, k * t["out"]:(k + 1) * t["out"]], ACT_RELU, ACT_NONE)
                     for k, (i, t) in enumerate(zip(ga.idx, ga.cfg["towers"]))]
            p2 = ob.opt_linear2_plan_create(descs, BF16, step.dev_index)
            gb.plan.launch(); gc.plan.launch(); p2.launch()
            torch.cuda.synchronize()
            same = bool(torch.equal(ref_out.view(torch.int16), out2.view(torch.int16)))
            flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device=device)

            def cold(fn, n=10):
                ts = []
                for _ in range(n):
                    flush.fill_(1)
                    c0, c1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    c0.record(stream); fn(); c1.record(stream)
                    torch.cuda.synchronize()
                    ts.append(c0.elapsed_time(c1) * 1e3)
                return float(np.mean(ts))
            # the whole tower in ONE launch: LayerNorm folded into the chain (opt_ln_linear2, reading Q25)
            out3 = torch.empty_like(ref_out)
            p3 = ob.opt_ln_linear2_plan_create(
                [ob.ln_linear2_member(T(i["x"]), T(i["gamma"]), T(i["beta"]), t["eps"], T(i["w1"]), T(i["b1"]), T(i["w2"]), T(i["b2"]),
                                      out3[:, k * t["out"]:(k + 1) * t["out"]], ACT_RELU, ACT_NONE)
                 for k, (i, t) in enumerate(zip(ga.idx, ga.cfg["towers"]))], BF16, step.dev_index)
            ga.plan.launch(); gb.plan.launch(); gc.plan.launch(); p3.launch()
            torch.cuda.synchronize()
            d3 = (out3.float() - ref_out.float())
            rel3 = float((d3.norm(dim=1) / ref_out.float().norm(dim=1).clamp_min(1e-30)).max())
            del d3
            t1 = cold(p2.launch)
            t5 = cold(p3.launch)
            t2 = cold(lambda: (gb.plan.launch(), gc.plan.launch()))
            t3 = cold(lambda: (ga.plan.launch(), p2.launch()))                       # whole C4 block: LN + chained Linear
            t4 = cold(lambda: (ga.plan.launch(), gb.plan.launch(), gc.plan.launch()))  # whole C4 block: three groups
            i2 = p2.info()
            vertical = dict(workload="C4 towers: Linear(D->H)+ReLU -> Linear(H->64), 512 members, B=8192", launches=1,
                            linear2_us=round(t1, 1), two_launch_us=round(t2, 1), speedup=round(t2 / t1, 3),
                            c4_block_ln_plus_linear2_us=round(t3, 1), c4_block_three_groups_us=round(t4, 1),
                            c4_block_one_launch_us=round(t5, 1), c4_block_one_launch_speedup=round(t4 / t5, 3),
                            c4_block_one_launch_bytes=p3.info()["bytes"],
                            c4_block_one_launch_row_l2_vs_three_groups=round(rel3, 5),
                            bitwise_equal_to_two_launch=same, flops=i2["flops"], algorithmic_bytes=i2["bytes"],
                            tflops=round(i2["flops"] / t1 / 1e6, 1),
                            frac_tensor=round(i2["flops"] / t1 / 1e6 / peaks["bf16_tflops"], 4),
                            hbm_bytes_saved=int(gb.info["bytes"] + gc.info["bytes"] - i2["bytes"]))
            del flush, out2, out3
        except Exception as e:  # noqa: BLE001
            vertical = dict(error=repr(e))

    # ---- (7) SURVEY 8(f) rank 3, side figure: backward of C2's grouped Linear through the same grouped kernel
    # (operands read in their stored layout, no transposed copies): one launch for all dgrads, one for all wgrads
    backward = None
    c2g = [g for g in step.groups if g.name.startswith("C2")]
    if c2g and not args.profile and not args.small:
        try:
            g2 = c2g[0]
            ycat = g2.aout.tensor(g2.iy)
            dy_cat = torch.empty_like(ycat).normal_(0.0, 1.0)
            dg, wg, keep = [], [], []
            for (ix, iw, ib), m in zip(g2.idx, g2.cfg["members"]):
                x, w = g2.ain.tensor(ix), g2.ain.tensor(iw)
                dy = dy_cat[:, m["col_off"]:m["col_off"] + m["N"]]
                dx, dw = torch.empty_like(x), torch.empty_like(w)
                keep.append((dx, dw))
                dg.append(ob.linear_member(dy, w, None, dx, ACT_NONE, ob.OPT_LAYOUT_W_TRANSPOSED))
                wg.append(ob.linear_member(dy, x, None, dw, ACT_NONE, ob.OPT_LAYOUT_X_TRANSPOSED | ob.OPT_LAYOUT_W_TRANSPOSED))
            pd, pw = ob.opt_linear_plan_create(dg, BF16, step.dev_index), ob.opt_linear_plan_create(wg, BF16, step.dev_index)
            flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device=device)

            def cold2(fn, n=10):
                ts = []
                for _ in range(n):
                    flush.fill_(1)
                    c0_, c1_ = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    c0_.record(stream); fn(); c1_.record(stream)
                    torch.cuda.synchronize()
                    ts.append(c0_.elapsed_time(c1_) * 1e3)
                return float(np.mean(ts))
            pd.launch(); pw.launch()
            torch.cuda.synchronize()
            td, tw_ = cold2(pd.launch), cold2(pw.launch)
            idg, iwg = pd.info(), pw.info()
            backward = dict(workload="configs[2] backward: dX = dY W and dW = dY^T X for the 128 members, one launch each",
                            dgrad_us=round(td, 1), dgrad_tflops=round(idg["flops"] / td / 1e6, 1),
                            wgrad_us=round(tw_, 1), wgrad_tflops=round(iwg["flops"] / tw_ / 1e6, 1),
                            frac_tensor_dgrad=round(idg["flops"] / td / 1e6 / peaks["bf16_tflops"], 4),
                            frac_tensor_wgrad=round(iwg["flops"] / tw_ / 1e6 / peaks["bf16_tflops"], 4))
            # bias gradients db = column sums of dY of the 128 members (slices of the concat gradient), one launch
            dbs = [torch.empty(m["N"], dtype=torch.float32, device=device) for m in g2.cfg["members"]]
            pb = ob.opt_bias_grad_plan_create([ob.bias_grad_member(dy_cat[:, m["col_off"]:m["col_off"] + m["N"]], d)
                                               for m, d in zip(g2.cfg["members"], dbs)], BF16, ob.OPT_F32, step.dev_index)
            pb.launch()
            torch.cuda.synchronize()
            tb_ = cold2(pb.launch)
            backward.update(bias_grad_workload="configs[2]: 128 bias gradients db = column sums of the members' slices of the [4096, sum N] concat gradient, one launch",
                            bias_grad_us=round(tb_, 1), bias_grad_gbs=round(pb.info()["bytes"] / tb_ / 1e3, 1),
                            bias_grad_frac_hbm=round(pb.info()["bytes"] / tb_ / 1e3 / peaks["hbm_gbs"], 4))
            # the whole backward of the group, three launches back to back in one timed region: ReLU mask fused into the
            # bias-gradient launch (dY and the stored output Y read, dZ written in place of dY, db summed), dgrads and
            # wgrads (which read dY's buffer, now holding dZ)
            pfb = ob.opt_bias_grad_plan_create([ob.bias_grad_member(dy_cat[:, m["col_off"]:m["col_off"] + m["N"]], d,
                                                                    ycat[:, m["col_off"]:m["col_off"] + m["N"]],
                                                                    dy_cat[:, m["col_off"]:m["col_off"] + m["N"]], ob.OPT_ACT_RELU)
                                                for m, d in zip(g2.cfg["members"], dbs)], BF16, ob.OPT_F32, step.dev_index)
            pfb.launch()
            torch.cuda.synchronize()
            tfb = cold2(pfb.launch)
            tall = cold2(lambda: (pfb.launch(), pd.launch(), pw.launch()))
            backward.update(whole_backward_workload="configs[2]: backward of the 128 Linear+bias+ReLU members in 3 launches (fused mask + bias gradient in place, dgrad, wgrad)",
                            relu_mask_bias_grad_fused_c2_us=round(tfb, 1), relu_mask_bias_grad_fused_c2_gbs=round(pfb.info()["bytes"] / tfb / 1e3, 1),
                            whole_backward_us=round(tall, 1), whole_backward_launches=3)
            del dbs
            # LayerNorm backward of C4a's 512 members (dx, dgamma, dbeta), one launch
            c4a = [g for g in step.groups if g.name.startswith("C4a")]
            if c4a:
                ga = c4a[0]
                lb, keep2 = [], []
                for i in ga.idx:
                    x, gam = ga.ain.tensor(i["x"]), ga.ain.tensor(i["gamma"])
                    dyl = torch.empty_like(x).normal_(0.0, 1.0)
                    dxl, dgl, dbl = torch.empty_like(x), torch.empty_like(gam), torch.empty_like(gam)
                    keep2.append((dyl, dxl, dgl, dbl))
                    lb.append(ob.layernorm_bwd_member(x, dyl, gam, dxl, dgl, dbl, 1e-5))
                pl = ob.opt_layernorm_bwd_plan_create(lb, BF16, BF16, step.dev_index)
                pl.launch()
                torch.cuda.synchronize()
                tl = cold2(pl.launch)
                il = pl.info()
                backward.update(layernorm_bwd_workload="configs[4] LayerNorm group backward (512 members, dx + dgamma + dbeta), one launch",
                                layernorm_bwd_us=round(tl, 1), layernorm_bwd_gbs=round(il["bytes"] / tl / 1e3, 1),
                                layernorm_bwd_frac_hbm=round(il["bytes"] / tl / 1e3 / peaks["hbm_gbs"], 4))
                del keep2
                # bias gradients of C4b's 512 Linear+ReLU members: column sums of a [B, H] gradient per member (the hidden
                # tensors stand in for dH: same shapes and layout), one launch
                db4 = [torch.empty(ga.amid.tensor(i["h"]).shape[1], dtype=torch.float32, device=device) for i in ga.idx]
                pb4 = ob.opt_bias_grad_plan_create([ob.bias_grad_member(ga.amid.tensor(i["h"]), d) for i, d in zip(ga.idx, db4)],
                                                   BF16, ob.OPT_F32, step.dev_index)
                pb4.launch()
                torch.cuda.synchronize()
                tb4 = cold2(pb4.launch)
                backward.update(bias_grad_c4_workload="configs[4] Linear+ReLU group: 512 bias gradients db = column sums of [8192, H], one launch",
                                bias_grad_c4_us=round(tb4, 1), bias_grad_c4_gbs=round(pb4.info()["bytes"] / tb4 / 1e3, 1),
                                bias_grad_c4_frac_hbm=round(pb4.info()["bytes"] / tb4 / 1e3 / peaks["hbm_gbs"], 4))
                # the same with the ReLU mask fused in front (dZ = dH-gradient where h > 0, written once, summed in the same pass)
                # against OPT_PW_RELU_BWD followed by the plain bias gradient
                gh = [torch.empty_like(ga.amid.tensor(i["h"])).normal_(0.0, 1.0) for i in ga.idx]
                dzs = [torch.empty_like(g_) for g_ in gh]
                pf4 = ob.opt_bias_grad_plan_create([ob.bias_grad_member(g_, d, ga.amid.tensor(i["h"]), z) for g_, d, i, z in zip(gh, db4, ga.idx, dzs)],
                                                   BF16, ob.OPT_F32, step.dev_index)
                pm4 = ob.opt_pointwise_plan_create([ob.chunk(g_, z, ob.OPT_PW_RELU_BWD, ga.amid.tensor(i["h"])) for g_, i, z in zip(gh, ga.idx, dzs)], BF16, step.dev_index)
                pz4 = ob.opt_bias_grad_plan_create([ob.bias_grad_member(z, d) for z, d in zip(dzs, db4)], BF16, ob.OPT_F32, step.dev_index)
                pf4.launch(); pm4.launch(); pz4.launch()
                torch.cuda.synchronize()
                tf4, tm4 = cold2(pf4.launch), cold2(lambda: (pm4.launch(), pz4.launch()))
                backward.update(relu_mask_bias_grad_fused_us=round(tf4, 1), relu_mask_bias_grad_fused_gbs=round(pf4.info()["bytes"] / tf4 / 1e3, 1),
                                relu_mask_bias_grad_fused_frac_hbm=round(pf4.info()["bytes"] / tf4 / 1e3 / peaks["hbm_gbs"], 4),
                                relu_mask_then_bias_grad_two_launches_us=round(tm4, 1))
                del db4, pb4, gh, dzs, pf4, pm4, pz4
                # activation_quantization_aten_pass: the 512 saved LayerNorm outputs -> FP8 E4M3 and back, one launch each
                A = ga.amid.tensor
                q8 = [torch.empty(A(i["xn"]).shape, dtype=torch.uint8, device=device) for i in ga.idx]
                r16 = [torch.empty_like(A(i["xn"])) for i in ga.idx]
                pq = ob.opt_pointwise_plan_create([ob.chunk(A(i["xn"]), q, ob.OPT_PW_QUANT_E4M3, None, [16.0])
                                                   for i, q in zip(ga.idx, q8)], BF16, step.dev_index)
                pdq = ob.opt_pointwise_plan_create([ob.chunk(q, r, ob.OPT_PW_DEQUANT_E4M3, None, [1.0 / 16.0])
                                                    for q, r in zip(q8, r16)], BF16, step.dev_index)
                pq.launch(); pdq.launch()
                torch.cuda.synchronize()
                tq, tdq = cold2(pq.launch), cold2(pdq.launch)
                backward.update(fp8_workload="configs[4] saved LayerNorm outputs (512 x [B, D] bf16) -> FP8 E4M3 and back, one launch each",
                                fp8_quant_us=round(tq, 1), fp8_quant_gbs=round(pq.info()["bytes"] / tq / 1e3, 1),
                                fp8_quant_frac_hbm=round(pq.info()["bytes"] / tq / 1e3 / peaks["hbm_gbs"], 4),
                                fp8_dequant_us=round(tdq, 1), fp8_dequant_gbs=round(pdq.info()["bytes"] / tdq / 1e3, 1),
                                fp8_dequant_frac_hbm=round(pdq.info()["bytes"] / tdq / 1e3 / peaks["hbm_gbs"], 4))
                del q8, r16
            del flush, keep, dy_cat
        except Exception as e:  # noqa: BLE001
            backward = dict(error=repr(e))

    # ---- (8) SURVEY 8(f) rank 4, side figure: the skinny aten.mm group of PAPER.md:477 (decompose_mm_pass), full size
    skinny = None
    if not args.profile and not args.small:
        try:
            shapes = [(18583840, 8, 8), (25247936, 4, 2), (22502112, 8, 8), (17980096, 4, 2)]       # (M, K, N)
            ten = [(torch.randn(M, K, device=device, dtype=torch.bfloat16), torch.randn(N, K, device=device, dtype=torch.bfloat16),
                    torch.empty(M, N, device=device, dtype=torch.bfloat16)) for M, K, N in shapes]
            ps = ob.opt_linear_plan_create([ob.linear_member(x, w, None, y, ACT_NONE) for x, w, y in ten], BF16, step.dev_index)
            flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device=device)

            def cold3(fn, n=5):
                ts = []
                for _ in range(n):
                    flush.fill_(1)
                    c0_, c1_ = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    c0_.record(stream); fn(); c1_.record(stream)
                    torch.cuda.synchronize()
                    ts.append(c0_.elapsed_time(c1_) * 1e3)
                return float(np.mean(ts))
            ps.launch()
            torch.cuda.synchronize()
            tsk = cold3(ps.launch)
            isk = ps.info()
            # the two [M,8]x[8,8] members alone: streaming row kernel vs the tensor-core tile kernel (opt_linear_options.no_skinny)
            two = [ob.linear_member(x, w, None, y, ACT_NONE) for (x, w, y), sh in zip(ten, shapes) if sh[1] == 8]
            p8 = ob.opt_linear_plan_create(two, BF16, step.dev_index)
            p8t = ob.opt_linear_plan_create_ex(two, BF16, step.dev_index, ob.opt_linear_options(no_skinny=1))
            p8.launch(); p8t.launch()
            torch.cuda.synchronize()
            t8, t8t = cold3(p8.launch), cold3(p8t.launch, 2)
            skinny = dict(workload="PAPER.md:477 model type B: aten.mm [18583840,8]x[8,8], [25247936,4]x[4,2], [22502112,8]x[8,8], "
                                   "[17980096,4]x[4,2] as ONE group, one launch (paper: each > 914 ms unfused on its hardware)",
                          launches=1, us=round(tsk, 1), algorithmic_bytes=isk["bytes"], gbs=round(isk["bytes"] / tsk / 1e3, 1),
                          frac_hbm=round(isk["bytes"] / tsk / 1e3 / peaks["hbm_gbs"], 4),
                          two_8x8_members_row_kernel_us=round(t8, 1), two_8x8_members_tensor_core_tiles_us=round(t8t, 1))
            del ten, flush
        except Exception as e:  # noqa: BLE001
            skinny = dict(error=repr(e))

    watch.stop_flag.set()
    watch.join(timeout=2)

    # max over ranks
    ms_total, ms_e2e, ms_e2e_ms = max_over_ranks([ms_total, ms_e2e, ms_e2e_ms], world, device)

    us_step = ms_total * 1e3 / K
    us_e2e = ms_e2e * 1e3 / Ke

    groups = {}
    for g, us, usmin in zip(step.groups, per_group_us, per_group_min_us):
        fl, by = g.info["flops"], g.info["bytes"]
        gbs = by / (us * 1e-6) / 1e9
        tfs = fl / (us * 1e-6) / 1e12
        t_hbm = by / (peaks["hbm_gbs"] * 1e9) * 1e6
        t_tc = fl / (peaks["bf16_tflops"] * 1e12) * 1e6
        groups[g.name] = dict(latency_us=round(us, 2), latency_min_us=round(usmin, 2), launches=1, tiles=g.info["tiles"],
                              algorithmic_bytes=by, flops=fl, gbs=round(gbs, 1), tflops=round(tfs, 1),
                              frac_hbm=round(gbs / peaks["hbm_gbs"], 4),
                              frac_tensor=round(tfs / peaks["bf16_tflops"], 4) if fl else None,
                              roofline_us=round(max(t_hbm, t_tc), 2),
                              frac_roofline=round(max(t_hbm, t_tc) / us, 4))
        if g.name in copy_ref:      # isolated, cold L2: this kernel next to torch's copy_ of the same byte count
            cus, kus = copy_ref[g.name]
            groups[g.name].update(isolated_cold_l2_us=round(kus, 2), same_size_copy_us=round(cus, 2),
                                  frac_of_same_size_copy=round(cus / kus, 4),
                                  isolated_frac_hbm=round(by / (kus * 1e-6) / 1e9 / peaks["hbm_gbs"], 4))

    # what north_star grades, per group, MEASURED in this run (CUDA events): in the step (power-capped, sustained
    # clocks) and isolated (cold L2, burst clocks).  HBM-bound groups against the measured copy bandwidth; configs[2]
    # (the "large-tower config", reading Q23) against the measured bf16 tensor peak -- burst for the isolated launch,
    # sustained for the in-step one -- with the roofline time as the per-member sum of max(tensor, HBM) next to it.
    per_group = {}
    for g, us in zip(step.groups, per_group_us):
        fl, by = g.info["flops"], g.info["bytes"]
        iso = isolated.get(g.name)
        d = dict(bound=g.bound, in_step_us=round(us, 2), isolated_us=None if iso is None else round(iso, 2))
        if g.bound == "hbm":
            d.update(frac_hbm_in_step=round(by / (us * 1e-6) / 1e9 / peaks["hbm_gbs"], 4),
                     frac_hbm_isolated=None if iso is None else round(by / (iso * 1e-6) / 1e9 / peaks["hbm_gbs"], 4))
            if g.name in copy_ref:
                d.update(same_size_copy_us=round(copy_ref[g.name][0], 2))
        else:
            d.update(frac_tensor_in_step_vs_sustained_peak=round(fl / (us * 1e-6) / 1e12 / peaks["bf16_tflops_sustained"], 4),
                     frac_tensor_in_step_vs_burst_peak=round(fl / (us * 1e-6) / 1e12 / peaks["bf16_tflops"], 4),
                     frac_tensor_isolated_vs_burst_peak=None if iso is None else round(fl / (iso * 1e-6) / 1e12 / peaks["bf16_tflops"], 4))
            ms_ = g.cfg["members"]
            t_sum = sum(max(2.0 * m["M"] * m["N"] * m["K"] / (peaks["bf16_tflops"] * 1e12),
                            2.0 * (m["M"] * m["K"] + m["N"] * m["K"] + m["N"] + m["M"] * m["N"]) / (peaks["hbm_gbs"] * 1e9)) for m in ms_) * 1e6
            t_roof = max(fl / (peaks["bf16_tflops"] * 1e12), by / (peaks["hbm_gbs"] * 1e9)) * 1e6
            d.update(roofline_us=round(t_roof, 2), roofline_per_member_sum_of_max_us=round(t_sum, 2),
                     frac_roofline_isolated=None if iso is None else round(t_roof / iso, 4),
                     frac_roofline_per_member_isolated=None if iso is None else round(t_sum / iso, 4))
        per_group[g.name] = d

    # dominant kernel of the step = the grouped GEMM (3 of the 6 launches); over a step it is HBM-bound
    # (C4b/C4c at 85 and 52 flop/B; C2 sits on the ridge and is reported against tensor peak in per_group)
    gemm = [(g, us) for g, us in zip(step.groups, per_group_us) if g.kind == "linear"]
    gemm_bytes = sum(g.info["bytes"] for g, _ in gemm)
    gemm_us = sum(us for _, us in gemm)
    achieved = gemm_bytes / (gemm_us * 1e-6) / 1e9
    traffic, traffic_note = (None, "debug sizes") if args.small else ncu_traffic_of_gemm_launches()
    roofline = dict(bound="hbm", kernel="grouped_gemm_sm100_kernel", achieved=round(achieved, 1), peak=peaks["hbm_gbs"],
                    unit="GB/s", frac=round(achieved / peaks["hbm_gbs"], 4),
                    traffic=traffic, traffic_source=traffic_note,
                    peak_source=peaks["source"] + ", burst copy figure",
                    launches_per_step=len(gemm), bytes_per_step=gemm_bytes, us_per_step=round(gemm_us, 2),
                    share_of_step=round(gemm_us / sum(per_group_us), 4), per_group=per_group)
    c2 = groups.get("C2_grouped_linear_tower")
    roofline_tensor = None
    if c2:
        roofline_tensor = dict(bound="tensor", kernel="grouped_gemm_sm100_kernel", workload="C2", achieved=c2["tflops"],
                               peak=peaks["bf16_tflops"], unit="TFLOP/s", frac=c2["frac_tensor"],
                               frac_of_sustained=round(c2["tflops"] / peaks["bf16_tflops_sustained"], 4))

    line = dict(metric="fused_op_group_step_latency", value=round(us_step, 2), unit="us", n_gpus=world, steps=K, warmup=W,
                ms_per_step=round(us_step / 1e3, 5), higher_is_better=False, scaling="weak", vs_baseline=None,
                dtype="bf16", data="synthetic",
                config=dict(workload=WORKLOAD_NAME if not args.small else "SMALL (debug sizes) " + json.dumps(SMALL),
                            parallelism="replicas x%d (no data-path collective)" % world,
                            l2="inputs larger than L2: a step touches %.2f GB, every group's data was last touched one "
                               "full step earlier" % (sum(g.info["bytes"] for g in step.groups) / 1e9),
                            groups_per_step=ng),
                e2e=dict(value=round(ms_e2e_ms * 1e3 / Ke, 2), unit="us", h2d_bytes_per_step=step.h2d_bytes(),
                         d2h_bytes_per_step=step.d2h_bytes(), steps=Ke, single_stream_us=round(us_e2e, 2),
                         api="opt_plan_launch_host (pinned host arenas; every input tensor H2D and every output D2H "
                             "each step); value: the four independent configs on four streams so that their PCIe "
                             "copies overlap, single_stream_us: everything on one stream"),
                gpu_launches=int(launches), launches_per_step=ng,
                clocks=watch.summary(), roofline=roofline, roofline_tensor=roofline_tensor, groups=groups,
                unfused_baseline=unfused, vertical_fusion=vertical, backward=backward, skinny_linear=skinny, config0_latency=c0,
                aggregate=dict(steps_per_s=round(aggregate_steps_per_s(us_step, world), 2)),
                build_seconds=round(build_s, 1), lib=ob.opt_version())

    if rank == 0 and not args.no_cpu and not args.profile and world >= 1:
        cfgs = {g.name[:2].lower(): g.cfg for g in step.groups}
        line["cpu_baseline"] = oracle_full_step(cfgs, small=args.small)
    if rank == 0:
        print(json.dumps(line))
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="product", choices=["product", "reference"])
    ap.add_argument("--e2e-steps", type=int, default=5)
    ap.add_argument("--small", action="store_true", help="debug sizes (not a bench number)")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--no-unfused", action="store_true", help="skip the one-launch-per-op baseline")
    ap.add_argument("--profile", action="store_true",
                    help="only the step's own launches (no cpu_baseline, no unfused baseline, no copy reference): for ncu")
    ap.add_argument("--ref-frac", type=float, default=0.0, help="reference arm: override the row-sample fraction")
    ap.add_argument("--side", default=None, choices=["linear2", "ln_linear2", "lhs", "skinny", "fp8", "fp8_fused", "bias_grad", "backward", "gemm_trace", "linear2_trace", "power"], help="stand-alone side workload for ncu (not the metric)")
    ap.add_argument("--ncu-summary", default=None, metavar="REP", help="CPU box: print the csv summary of an ncu --set full capture of `bench.py --profile`")
    args = ap.parse_args()
    if args.ncu_summary:
        return write_ncu_summary(args.ncu_summary)
    if args.side:
        return run_side(args)
    if args.impl == "reference":
        return run_reference(args)
    return run_product(args)


if __name__ == "__main__":
    sys.exit(main())
