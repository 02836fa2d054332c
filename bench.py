#!/usr/bin/env python
"""bench.py -- throughput of the hot path on B200(s), one JSON line on stdout.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload NAME] [--suite primary|baseline|full]
    python bench.py --impl reference ...        # the CPU oracle on the host cores
    python bench.py --fig1                      # the paper's Fig. 1 on this GPU (not a benchmark line)

A "step" is one pass of the hot path over one batch of the named workload (seeded,
synthetic -- this path has no dataset): for the default workload C2 (the config
BASELINE.json's metric is quoted on, Philox4x32-10, 2^20 streams x 1024 u32 = 4 GiB)
that is one rng_fill_u32 call.  `value` is whole-job throughput with the output
resident in HBM; `e2e` is the same metric through the host-buffer C-ABI call
(rng_fill_u32_host into pinned host memory, device->host copy inside the timed region).
The stdout line is ONE compact JSON object (< 4 KB, tests/test_bench_contract.py).  `--suite
baseline` (default at N=1 for the default workload) also measures BASELINE.json's other configs
(C1, C2 f32, C3, C4, C5b) and adds them as `"configs"`: rows of [workload, value, unit,
roofline frac]; `--suite full` measures every workload of the registry.  Per-workload detail goes
to stderr (one short line each) and, with `--dump PATH`, as a JSON list to that file.
`config.workload` is the same short name (`--workload`) in both arms.  See DESIGN.md section 7.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_1204_6193_b200 import workloads as W  # noqa: E402  (plain data, no arithmetic)

METRIC = "Gnum/s per generator (HBM-fill & in-register modes); Ising spin flips/ns"


def log(*a):
    print(*a, file=sys.stderr, flush=True)


def measured_peaks() -> dict:
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return {"hbm_gbs": float(d["hbm_gbs"]), "sm_max_mhz": float(d.get("sm_max_mhz", 1965.0)), "source": "measured"}
    # fallback stated in /opt/skills/guides/B200_PROFILING.md
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0, "source": "fallback"}


N_SM, SMSP_PER_SM, LANES = 148, 4, 32  # B200: 148 SMs x 4 schedulers x 1 warp-instruction/clk


TRAFFIC_JSON = os.path.join(ROOT, "profiles", "traffic.json")


def _capture(name: str):
    """the workload's entry of profiles/traffic.json: figures of its dominant kernel from the committed
    `ncu --set full` capture (written by `python tests/ncu_summary.py` from ncu's raw page).
    STATIC: captured in an earlier run of the same command under ncu, never measured in the run that prints it."""
    try:
        return json.load(open(TRAFFIC_JSON)).get(name)
    except Exception:
        return None


def measured_traffic(name: str):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel (static capture)"""
    e = _capture(name)
    return e.get("dram_bytes_per_launch") if e else None


PIPES = ("alu", "fma", "fmaheavy", "lsu")


def measured_ncu(name: str):
    """ncu-measured utilisation of the workload's dominant kernel (static capture): issue slots, the busiest
    pipe and its utilisation, DRAM throughput; None if this workload was not captured"""
    e = _capture(name)
    if not e:
        return None
    pipes = {"alu": e.get("pipe_alu_pct"), "fma": e.get("pipe_fma_pct"), "lsu": e.get("pipe_lsu_pct"),
             "fmaheavy": e.get("pipe_fmaheavy_cycles_pct_of_elapsed")}
    pipes = {k: v for k, v in pipes.items() if v is not None}
    top = max(pipes, key=pipes.get) if pipes else None
    r1 = lambda v: None if v is None else round(float(v), 1)  # noqa: E731
    return {"issue_active_pct": r1(e.get("issue_active_pct")), "binding_pipe": top,
            "binding_pipe_pct": r1(pipes.get(top)) if top else None,
            "dram_throughput_pct": r1(e.get("dram_throughput_pct")), "time_us": e.get("ncu_time_us"),
            "kernel": (e.get("kernel") or "").replace("void ", "").split("(")[0],
            "capture": e.get("source"), "measured_in_this_run": False}


def issue_peak_tinst(sm_mhz: float) -> float:
    """thread-instruction issue peak in Tinst/s ('alu' roofline)"""
    return N_SM * SMSP_PER_SM * LANES * sm_mhz * 1e6 / 1e12


# algorithmic thread-instructions per draw (DESIGN.md section 7 derives each count from the
# recurrences as written in the paper, not from the compiled SASS): LCG64 = 64-bit multiply-add
# in 32-bit pieces (3) + checksum (2); XORWOW = 3 shifts + 3 xors + 2 adds + checksum (2);
# Philox = per word 5 mulhi/lo + 5 xors + key/counter (2); xs1024 register-resident = 66 funnel
# shifts + 66 xors per 32 words (the zero padding drops 10 of 32 words per phase) + Weyl add (1)
# + checksum (2)
ALG_INST_PER_DRAW = {W.LCG64: 5.0, W.LCG64_LEAPFROG: 5.0, W.XORWOW: 10.0, W.PHILOX4X32_10: 12.0, W.XS1024W: 7.0,
                     W.PHILOX4X32_7: 9.0, W.LCG32: 3.0, W.XS1024W_SKIP: 7.0,
                     W.LCG64_BOTH: 3.5, W.LFIB521: 8.0, W.LFIB1279: 8.0, W.LCG32_LEAPFROG: 3.0, W.MWC: 3.0, W.MWC_MULTI: 3.0}  # lfib: 2 LDS, add, compare-subtract, STS,
# barrier, 2 checksum
# multi-spin-coded update: two threshold compares of two instructions each + the bit-sliced
# neighbour count / flip logic amortised over the 32 sites of a word (about 1), excl. the draw
ALG_INST_PER_ISING_UPDATE = 5.0
STATE_BYTES = {W.LCG64: 8, W.LCG64_LEAPFROG: 8, W.XORWOW: 24, W.PHILOX4X32_10: 0, W.XS1024W: 4, W.PHILOX4X32_7: 0,
               W.LCG32: 4, W.XS1024W_SKIP: 4, W.LCG64_BOTH: 8,
               W.LFIB521: 521 * 4 / 256.0, W.LFIB1279: 1279 * 4 / 256.0, W.LCG32_LEAPFROG: 4, W.MWC: 8, W.MWC_MULTI: 10}


# The paper's own numbers (GTX 480) for the workloads that have one: context, not a target.
# Table 2: peak 10^9 numbers/s consumed in-register; Table 1: 1/t_up flips/ns
# of the double-checkerboard code at L = 1024, beta = 0.4.
PAPER_GTX480 = {
    "C3_xorwow_2^22x256_draw_reduce": (19.0, "Gnum/s", "PAPER.md:266"),
    "C4_xs1024_2^24x4096_draw_draw_reduce": (18.0, "Gnum/s", "PAPER.md:268"),
    "N1_philox10_2^22x256_draw_reduce": (30.0, "Gnum/s", "PAPER.md:270"),
    "N1_philox7_2^22x256_draw_reduce": (41.0, "Gnum/s", "PAPER.md:269"),
    "N1_lcg64_2^22x256_draw_reduce": (46.0, "Gnum/s", "PAPER.md:261"),
    "N1_lcg32_2^22x256_draw_reduce": (58.0, "Gnum/s", "PAPER.md:259"),
    "N3_mwc_2^22x256_draw_reduce": (44.0, "Gnum/s", "PAPER.md:95, :263"),
    "T1_multihit_L1024_mwc_k100": (1.0 / 0.0435, "flips/ns", "PAPER.md:84"),
    "T1_multihit_L1024_lfib521_k100": (1.0 / 0.0661, "flips/ns", "PAPER.md:86"),
    "T1_multihit_L1024_lfib1279_k100": (1.0 / 0.0700, "flips/ns", "PAPER.md:87"),
    "N4_lfib521_2^22x256_draw_reduce": (23.0, "Gnum/s", "PAPER.md:264"),
    "N4_lfib1279_2^22x256_draw_reduce": (23.0, "Gnum/s", "PAPER.md:265"),
    "T1_multihit_L1024_xorwow_k1": (1.0 / 0.7956, "flips/ns", "PAPER.md:88"),
    "T1_multihit_L1024_xorwow_k100": (1.0 / 0.0576, "flips/ns", "PAPER.md:88"),
    "T1_multihit_L1024_xorwow_k100_tile8": (1.0 / 0.0576, "flips/ns", "PAPER.md:88"),
    "T1_multihit_L1024_philox_k100": (1.0 / 0.0622, "flips/ns", "PAPER.md:91"),
    "T1_multihit_L1024_xs1024skip_k100": (1.0 / 0.0721, "flips/ns", "PAPER.md:89"),
    "T1_multihit_L1024_lcg32_k100": (1.0 / 0.0402, "flips/ns", "PAPER.md:80"),
}


class ClockSampler:
    """samples SM clock and throttle reasons with NVML while the timed region runs"""

    def __init__(self, index: int, period_s: float = 0.001):
        self.index, self.period, self.samples, self.reasons = index, period_s, [], set()
        self._stop = threading.Event()
        self._thr = None
        self.max_mhz = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
        except Exception as e:  # pragma: no cover
            log(f"[bench] NVML unavailable: {e}")
            self.nv = None

    _NAMES = {0x1: "gpu_idle", 0x2: "applications_clocks_setting", 0x4: "sw_power_cap", 0x8: "hw_slowdown",
              0x10: "sync_boost", 0x20: "sw_thermal_slowdown", 0x40: "hw_thermal_slowdown",
              0x80: "hw_power_brake_slowdown", 0x100: "display_clock_setting"}

    def _run(self):
        nv = self.nv
        while not self._stop.is_set():
            try:
                self.samples.append(float(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                r = int(nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)) if hasattr(
                    nv, "nvmlDeviceGetCurrentClocksEventReasons") else int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
                for bit, name in self._NAMES.items():
                    if r & bit and name != "gpu_idle":
                        self.reasons.add(name)
            except Exception:
                pass
            self._stop.wait(self.period)

    def start(self):
        if self.nv:
            self._thr = threading.Thread(target=self._run, daemon=True)
            self._thr.start()

    def stop(self) -> dict:
        self._stop.set()
        if self._thr:
            self._thr.join()
        s = sorted(self.samples)
        med = s[len(s) // 2] if s else None
        return {"sm_mhz": med, "sm_min_mhz": s[0] if s else None, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(s), "sample_period_ms": self.period * 1e3}


# ------------------------------------------------------------------------------------
# jobs: what one step of each workload is, and the roofline that bounds its kernel
# ------------------------------------------------------------------------------------
class Job:
    """one workload on this rank's GPU; step() enqueues one step on the current stream"""
    name = ""
    unit = "Gnum/s"
    dtype = "u32"
    bound = "hbm"

    def units_per_step(self) -> float: ...
    def step(self): ...
    def alg_per_launch(self) -> float: ...   # bytes (hbm) or thread-instructions (alu) per kernel launch
    def close(self): ...


class FillJob(Job):
    def __init__(self, cfg: W.FillCfg, f32: bool, rank: int, world: int, out_buf):
        import paper_1204_6193_b200 as pkg
        from paper_1204_6193_b200.sharding import weak_scaling_shard
        self.cfg, self.f32 = cfg, f32
        self.name = cfg.name + ("_f32" if f32 else "_u32")
        n_total, first, n_local = weak_scaling_shard(rank, world, cfg.n_streams)
        self.rng = pkg.Rng(cfg.kind, n_local, cfg.seed, first=first, n_total=n_total)
        self.out = out_buf
        assert out_buf.numel() >= cfg.draws_per_call
        self.fn = self.rng.fill_f32 if f32 else self.rng.fill_u32
        self.dtype = "f32" if f32 else "u32"

    def units_per_step(self):
        return float(self.cfg.draws_per_call * self.cfg.calls)

    def step(self):
        for _ in range(self.cfg.calls):
            self.fn(self.out, self.cfg.n_per_stream)

    def alg_per_launch(self):
        # 4 B written per draw + one state load and one state store per stream per launch
        return 4.0 * self.cfg.draws_per_call + 2.0 * STATE_BYTES[self.cfg.kind] * self.cfg.n_streams

    def close(self):
        self.rng.close()


class DrawJob(Job):
    bound = "alu"

    def __init__(self, cfg: W.FillCfg, rank: int, world: int, out_buf):
        import paper_1204_6193_b200 as pkg
        from paper_1204_6193_b200.sharding import weak_scaling_shard
        self.cfg = cfg
        self.name = cfg.name + "_draw_reduce"
        n_total, first, n_local = weak_scaling_shard(rank, world, cfg.n_streams)
        self.rng = pkg.Rng(cfg.kind, n_local, cfg.seed, first=first, n_total=n_total)
        self.out = out_buf
        assert out_buf.numel() >= 2 * cfg.n_streams

    def units_per_step(self):
        return float(self.cfg.draws_per_call)

    def step(self):
        self.rng.draw_reduce(self.out, self.cfg.n_per_stream)

    def alg_per_launch(self):
        return ALG_INST_PER_DRAW[self.cfg.kind] * self.cfg.draws_per_call

    def close(self):
        self.rng.close()


class SeedJob(Job):
    """row a1: one step = rng_create (allocate + seed every stream; synchronous) + rng_destroy.
    Unit: streams seeded per second.  Bound by launch count and allocation for the random
    seeding, by the vector-matrix products for the paper's skip-ahead."""
    bound = "alu"
    unit = "Gstreams/s"
    dtype = "u32"

    def __init__(self, name: str, kind: int, n_streams: int, rank: int, world: int):
        from paper_1204_6193_b200.sharding import weak_scaling_shard
        self.name, self.kind = name, kind
        self.n_total, self.first, self.n_local = weak_scaling_shard(rank, world, n_streams)

    def units_per_step(self):
        return float(self.n_local)

    def step(self):
        import paper_1204_6193_b200 as pkg
        pkg.Rng(self.kind, self.n_local, W.MASTER_SEED, first=self.first, n_total=self.n_total).close()

    def alg_per_launch(self):
        # skip-ahead: one vector-matrix product per instance = 1024 predicated loads + 512 xors (average) per
        # 32 streams; random seeding: 16 splitmix64 outputs of ~10 instructions per instance
        per_inst = 1536.0 * 32 if self.kind == W.XS1024W_SKIP else 160.0
        return per_inst * self.n_local / 32.0

    def close(self):
        pass


class IsingJob(Job):
    bound = "alu"
    unit = "flips/ns"
    dtype = "int8"

    def __init__(self, cfg: W.IsingCfg, rank: int, world: int, sweeps_per_step: int):
        import torch
        import paper_1204_6193_b200 as pkg
        from paper_1204_6193_b200.sharding import weak_scaling_shard
        self.cfg, self.sweeps = cfg, sweeps_per_step
        self.name = cfg.name
        # replicas: every rank sweeps its own L x L lattice with its own stream block
        n_total, first, n_local = weak_scaling_shard(rank, world, cfg.n_streams)
        self.rng = pkg.Rng(cfg.kind, n_local, cfg.seed, first=first, n_total=n_total)
        self.spins = torch.empty(cfg.L * cfg.L, dtype=torch.int8, device="cuda")
        pkg.ising_init_random(self.spins, cfg.L, cfg.lattice_seed + rank)
        # a half-sweep launch loads and stores every stream's state once: with few updates per
        # stream (the paper's k = 1 regime) that traffic, not the arithmetic, bounds the kernel
        self.K = cfg.L * cfg.L // 2 // cfg.n_streams if not cfg.tile else 2 * cfg.k_hits  # draws per state load
        self.state_bytes_per_update = 2.0 * STATE_BYTES[cfg.kind] / self.K
        if self.state_bytes_per_update >= 4.0:
            self.bound = "hbm"

    def units_per_step(self):
        return float(self.cfg.L * self.cfg.L * self.sweeps * self.cfg.k_hits)

    def step(self):
        if self.cfg.tile:
            self.rng.ising_sweep_multihit(self.spins, self.cfg.L, self.cfg.beta, self.sweeps, self.cfg.tile,
                                          self.cfg.k_hits)
        else:
            self.rng.ising_sweep(self.spins, self.cfg.L, self.cfg.beta, self.sweeps)

    def alg_per_launch(self):
        k = self.cfg.L * self.cfg.L // 2  # updates per half-sweep launch
        if self.cfg.tile:
            # one launch = one coarse colour: half the sites, k_hits updates each; byte lattice, one generator
            # state load + store per thread.  ~12 instructions per update on bytes in shared memory + the draw
            if self.bound == "hbm":
                return 2.0 * STATE_BYTES[self.cfg.kind] * self.cfg.n_streams + 2.0 * k
            return (12.0 + ALG_INST_PER_DRAW[self.cfg.kind]) * k * self.cfg.k_hits
        if self.bound == "hbm":
            # state load + store per stream, plus the two bit planes read and one written (1 bit per site)
            return 2.0 * STATE_BYTES[self.cfg.kind] * self.cfg.n_streams + 3.0 * k / 8.0
        return (ALG_INST_PER_ISING_UPDATE + ALG_INST_PER_DRAW[self.cfg.kind]) * k

    def close(self):
        self.rng.close()


def max_over_ranks(ms: float) -> float:
    """the slowest rank's time (the contract's max over ranks); the tensor lives where the backend reduces: on
    the GPU for nccl, on the host for gloo (the CPU-side rendezvous test of the N > 1 flow)"""
    import torch
    dist = torch.distributed
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor([ms], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def roofline(name: str, bound: str, alg_per_launch: float, sec_per_launch: float, store_gbs=None) -> dict:
    """the `roofline` object of one workload.  hbm: algorithmic bytes per launch / measured launch duration against
    the measured copy bandwidth (MEASURED_PEAKS.json), and against the live write-only (memset) ceiling of this run
    when it was probed (a fill only writes; a copy reads and writes).  alu: the ncu-measured issue-slot and
    binding-pipe utilisation lead (static capture); achieved/peak/frac are the hand-counted algorithmic
    thread-instructions against the issue-slot peak, tagged as such."""
    peaks = measured_peaks()
    ncu = measured_ncu(name)
    if bound == "hbm":
        ach = alg_per_launch / sec_per_launch / 1e9
        r = {"bound": "hbm", "achieved": round(ach, 1), "peak": peaks["hbm_gbs"], "unit": "GB/s",
             "frac": round(ach / peaks["hbm_gbs"], 4), "traffic": measured_traffic(name),
             "algorithmic_bytes": int(alg_per_launch), "peak_source": peaks["source"] + " copy bandwidth"}
        if store_gbs:
            r["store_ceiling"] = round(store_gbs, 1)
            r["frac_vs_store_ceiling"] = round(ach / store_gbs, 4)
    else:
        ach = alg_per_launch / sec_per_launch / 1e12
        peak = issue_peak_tinst(peaks["sm_max_mhz"])
        # north_star asks for the ncu-MEASURED fraction of the issue peak: `frac` is smsp__issue_active of the
        # committed capture of this workload's kernel (a static figure, not of this run); the hand-counted
        # algorithmic instructions against the same peak are kept beside it as frac_algorithmic
        r = {"bound": "alu", "achieved": round(ach, 3), "peak": round(peak, 3), "unit": "Tinst/s",
             "frac": round(ach / peak, 4), "frac_algorithmic": round(ach / peak, 4),
             "basis": "algorithmic instruction count", "traffic": measured_traffic(name),
             "peak_source": "148 SM x 4 SMSP x 32 lanes x sm_max_mhz issue slots"}
        if ncu and ncu["issue_active_pct"] is not None:
            r["frac"] = round(ncu["issue_active_pct"] / 100.0, 4)
            r["basis"] = "frac = ncu smsp__issue_active (committed capture); achieved and frac_algorithmic = algorithmic instruction count"
            r["ncu_issue_active_pct"] = ncu["issue_active_pct"]
            r["ncu_binding_pipe"] = f"{ncu['binding_pipe']} {ncu['binding_pipe_pct']}%"
    r["ncu"] = ncu
    return r


def run_job(job: Job, steps: int, warmup: int, world: int, sample_clocks: bool, dev_index: int,
            store_gbs=None) -> dict:
    """W untimed warm-up steps, then EXACTLY `steps` steps between barrier+synchronize,
    timed with CUDA events on the launching stream; max over ranks."""
    import torch
    import paper_1204_6193_b200 as pkg
    dist = torch.distributed if world > 1 else None
    for _ in range(warmup):
        job.step()
    torch.cuda.synchronize()
    if dist:
        dist.barrier()
    sampler = ClockSampler(dev_index) if sample_clocks else None
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    l0 = pkg.rng_kernel_launches()
    if sampler:
        sampler.start()
    torch.cuda.synchronize()
    ev0.record()
    for _ in range(steps):
        job.step()
    ev1.record()
    torch.cuda.synchronize()
    clocks = sampler.stop() if sampler else None
    launches = pkg.rng_kernel_launches() - l0
    ms = ev0.elapsed_time(ev1)
    if dist:
        ms = max_over_ranks(ms)
        dist.barrier()
    units = job.units_per_step() * steps * world
    per_s = units / (ms * 1e-3)
    value = per_s / 1e9  # Gnum/s, and flips/ns == 1e9 flips/s
    res = {"name": job.name, "value": value, "unit": job.unit, "steps": steps, "warmup": warmup,
           "ms_per_step": ms / steps, "gpu_launches": int(launches), "dtype": job.dtype}
    # roofline of the (single) dominant kernel: average launch duration = timed region / launches
    n_l = steps if isinstance(job, SeedJob) else max(int(launches), 1)  # SeedJob counts per step (many small launches)
    res["roofline"] = roofline(getattr(job, "key", job.name), job.bound, job.alg_per_launch(), ms * 1e-3 / n_l, store_gbs)
    if clocks:
        res["clocks"] = clocks
    if job.name in PAPER_GTX480:
        v, u, cite = PAPER_GTX480[job.name]
        res["paper_gtx480"] = {"value": v, "unit": u, "cite": cite, "ratio": value / v,
                               "note": "the paper's number on its GTX 480: context, not the target"}
    return res


# ------------------------------------------------------------------------------------
# workload registry
# ------------------------------------------------------------------------------------
def make_job(name: str, rank: int, world: int, buf, ising_sweeps: int) -> Job:
    table = {
        "C2_u32": lambda: FillJob(W.C2, False, rank, world, buf),
        "C2_f32": lambda: FillJob(W.C2, True, rank, world, buf),
        "C1_u32": lambda: FillJob(W.C1, False, rank, world, buf),
        "C1_f32": lambda: FillJob(W.C1, True, rank, world, buf),
        "C1big_u32": lambda: FillJob(W.C1_BIG, False, rank, world, buf),
        "C3fill_u32": lambda: FillJob(W.C3_FILL, False, rank, world, buf),
        "N1_philox7_u32": lambda: FillJob(W.N1_PHILOX7, False, rank, world, buf),
        "N1_lcg32_u32": lambda: FillJob(W.N1_LCG32, False, rank, world, buf),
        "N1_philox7_draw": lambda: DrawJob(W.N1_PHILOX7_DRAW, rank, world, buf),
        "N1_philox10_draw": lambda: DrawJob(W.N1_PHILOX10_DRAW, rank, world, buf),
        "N1_lcg32_draw": lambda: DrawJob(W.N1_LCG32_DRAW, rank, world, buf),
        "N1_lcg64_draw": lambda: DrawJob(W.N1_LCG64_DRAW, rank, world, buf),
        "N1_lcg64both_draw": lambda: DrawJob(W.N1_LCG64BOTH_DRAW, rank, world, buf),
        "N3_mwc_draw": lambda: DrawJob(W.N3_MWC_DRAW, rank, world, buf),
        "T1_mwc_k100": lambda: IsingJob(W.T1_MWC_K100, rank, world, W.T1_MWC_K100.n_sweeps),
        "T1_lfib521_k100": lambda: IsingJob(W.T1_LFIB521_K100, rank, world, W.T1_LFIB521_K100.n_sweeps),
        "T1_lfib1279_k100": lambda: IsingJob(W.T1_LFIB1279_K100, rank, world, W.T1_LFIB1279_K100.n_sweeps),
        "N1_lcg64both_u32": lambda: FillJob(W.N1_LCG64BOTH, False, rank, world, buf),
        "N4_lfib521_f32": lambda: FillJob(W.N4_LFIB521, True, rank, world, buf),
        "N4_lfib1279_f32": lambda: FillJob(W.N4_LFIB1279, True, rank, world, buf),
        "N4_lfib521_draw": lambda: DrawJob(W.N4_LFIB521_DRAW, rank, world, buf),
        "N4_lfib1279_draw": lambda: DrawJob(W.N4_LFIB1279_DRAW, rank, world, buf),
        "C3_draw": lambda: DrawJob(W.C3, rank, world, buf),
        "C4_fill": lambda: FillJob(W.C4_FILL, False, rank, world, buf),
        "C4_draw": lambda: DrawJob(W.C4_DRAW, rank, world, buf),
        "N2_seed_xs1024_random": lambda: SeedJob("N2_seed_xs1024_random_2^24", W.XS1024W, 1 << 24, rank, world),
        "N2_seed_xs1024_skip": lambda: SeedJob("N2_seed_xs1024_skip_2^24", W.XS1024W_SKIP, 1 << 24, rank, world),
        "C5b_philox": lambda: IsingJob(W.C5B_PHILOX, rank, world, ising_sweeps),
        "C5b_xorwow": lambda: IsingJob(W.C5B_XORWOW, rank, world, ising_sweeps),
        "C5b_xorwow_K8": lambda: IsingJob(W.C5B_XORWOW_K8, rank, world, ising_sweeps),
        "T1_xorwow_k1": lambda: IsingJob(W.T1_XORWOW_K1, rank, world, W.T1_XORWOW_K1.n_sweeps),
        "T1_xorwow_k100": lambda: IsingJob(W.T1_XORWOW_K100, rank, world, W.T1_XORWOW_K100.n_sweeps),
        "T1_philox_k100": lambda: IsingJob(W.T1_PHILOX_K100, rank, world, W.T1_PHILOX_K100.n_sweeps),
        "T1_xs1024skip_k100": lambda: IsingJob(W.T1_XS1024_K100, rank, world, W.T1_XS1024_K100.n_sweeps),
        "T1_lcg32_k100": lambda: IsingJob(W.T1_LCG32_K100, rank, world, W.T1_LCG32_K100.n_sweeps),
        "T1big_xorwow_k100": lambda: IsingJob(W.T1BIG_XORWOW_K100, rank, world, W.T1BIG_XORWOW_K100.n_sweeps),
        "T1big_xorwow_k1": lambda: IsingJob(W.T1BIG_XORWOW_K1, rank, world, W.T1BIG_XORWOW_K1.n_sweeps),
        "T1big_xorwow_k100_t8": lambda: IsingJob(W.T1BIG_XORWOW_K100_T8, rank, world, W.T1BIG_XORWOW_K100_T8.n_sweeps),
        "T1_xorwow_k100_t8": lambda: IsingJob(W.T1_XORWOW_K100_T8, rank, world, W.T1_XORWOW_K100_T8.n_sweeps),
    }
    if name not in table:
        raise SystemExit(f"unknown --workload {name}; choose from {sorted(table)}")
    job = table[name]()
    job.key = name  # the --workload name: what config.workload and profiles/traffic.json are keyed by
    return job


# (name, steps, warmup): the secondary configs of --suite full; sized so that the whole
# default run stays within a few minutes
SUITE = [("C2_f32", 20, 3), ("C1_u32", 1000, 20), ("C1_f32", 1000, 20), ("C1big_u32", 20, 3), ("C3fill_u32", 20, 3),
         ("C3_draw", 20, 3), ("C4_fill", 3, 1), ("C4_draw", 1, 1), ("C5b_philox", 1, 1), ("C5b_xorwow", 1, 1),
         ("C5b_xorwow_K8", 1, 1),
         ("N1_philox7_u32", 20, 3), ("N1_lcg32_u32", 20, 3), ("N1_philox7_draw", 20, 3), ("N1_philox10_draw", 20, 3),
         ("N1_lcg32_draw", 20, 3), ("N1_lcg64_draw", 20, 3), ("N1_lcg64both_draw", 20, 3), ("N1_lcg64both_u32", 20, 3), ("N3_mwc_draw", 20, 3), ("T1_mwc_k100", 3, 3), ("T1_lfib521_k100", 3, 3), ("T1_lfib1279_k100", 3, 3),
         ("N4_lfib521_f32", 20, 3), ("N4_lfib1279_f32", 20, 3), ("N4_lfib521_draw", 20, 3), ("N4_lfib1279_draw", 20, 3),
         ("N2_seed_xs1024_random", 5, 3), ("N2_seed_xs1024_skip", 5, 3),
         ("T1_xorwow_k1", 3, 3), ("T1_xorwow_k100", 3, 3), ("T1_philox_k100", 3, 3), ("T1_xs1024skip_k100", 3, 3),
         ("T1_lcg32_k100", 3, 3), ("T1big_xorwow_k100", 3, 3), ("T1big_xorwow_k1", 3, 3),
         ("T1_xorwow_k100_t8", 3, 3), ("T1big_xorwow_k100_t8", 3, 3)]


# ------------------------------------------------------------------------------------
# the CPU oracle legs (the only places bench.py executes oracle/)
# ------------------------------------------------------------------------------------
def oracle_sample_rate(workload: str, target_s: float = 4.0, threads: int | None = None) -> dict:
    """time the oracle, as it stands, on a bounded sample of the workload on all host cores (or on `threads`
    of them: the oracle's only concession to run time is `omp parallel for` over independent streams, and
    orc_set_threads(1) turns that off); returns {"value","unit","cores","kind","sample","seconds"}"""
    import oracle
    if threads is not None:
        all_cores = oracle.threads()
        oracle.set_threads(threads)
        try:
            return oracle_sample_rate(workload, target_s)
        finally:
            oracle.set_threads(all_cores)
    cores = oracle.threads()
    if workload.startswith("T1"):
        cfg = {"T1_xorwow_k1": W.T1_XORWOW_K1, "T1_xorwow_k100": W.T1_XORWOW_K100, "T1_philox_k100": W.T1_PHILOX_K100,
               "T1_xs1024skip_k100": W.T1_XS1024_K100, "T1_lcg32_k100": W.T1_LCG32_K100, "T1_mwc_k100": W.T1_MWC_K100,
               "T1_lfib521_k100": W.T1_LFIB521_K100, "T1_lfib1279_k100": W.T1_LFIB1279_K100,
               "T1big_xorwow_k100": W.T1BIG_XORWOW_K100, "T1big_xorwow_k1": W.T1BIG_XORWOW_K1,
               "T1big_xorwow_k100_t8": W.T1BIG_XORWOW_K100_T8, "T1_xorwow_k100_t8": W.T1_XORWOW_K100_T8}[workload]
        L = 1024  # the paper's lattice; for the L = 8192 workloads 1/64 of the area, same tile and hits
        sp = oracle.ising_init_random(L, cfg.lattice_seed)
        r = oracle.Rng(cfg.kind, L * L // 4, cfg.seed)
        sweeps, t0 = 0, time.perf_counter()
        while True:
            r.ising_sweep_multihit(sp, L, cfg.beta, 1, cfg.tile, cfg.k_hits)
            sweeps += 1
            dt = time.perf_counter() - t0
            if dt > target_s or sweeps >= 1000:
                break
        return {"value": L * L * sweeps * cfg.k_hits / dt / 1e9, "unit": "flips/ns", "cores": cores, "kind": "oracle",
                "sample": f"L={L}, tile {cfg.tile}, k={cfg.k_hits}, {sweeps} sweeps", "seconds": dt}
    if workload.startswith("C5b"):
        cfg = {"C5b_philox": W.C5B_PHILOX, "C5b_xorwow": W.C5B_XORWOW, "C5b_xorwow_K8": W.C5B_XORWOW_K8}[workload]
        L = 2048  # 1/16 of the lattice area, same K per stream
        S = cfg.n_streams // 16
        sp = oracle.ising_init_random(L, cfg.lattice_seed)
        r = oracle.Rng(cfg.kind, S, cfg.seed)
        sweeps, t0 = 0, time.perf_counter()
        while True:
            r.ising_sweep(sp, L, cfg.beta, 1)
            sweeps += 1
            dt = time.perf_counter() - t0
            if dt > target_s or sweeps >= 1000:
                break
        return {"value": L * L * sweeps / dt / 1e9, "unit": "flips/ns", "cores": cores, "kind": "oracle",
                "sample": f"L={L} (1/16 of the 8192^2 lattice, same sites per stream), {sweeps} sweeps", "seconds": dt}
    if workload.startswith("N2_seed"):
        kind = oracle.XS1024W_SKIP if workload.endswith("skip") else oracle.XS1024W
        n_streams, S = 1 << 24, 1 << 12
        while True:  # seeding = creating the oracle's generator; grow the sample until it takes about target_s
            t0 = time.perf_counter()
            oracle.Rng(kind, S, W.MASTER_SEED)
            dt = max(time.perf_counter() - t0, 1e-6)
            if dt > target_s / 2 or S >= n_streams:
                break
            S = min(n_streams, S * 4)
        return {"value": S / dt / 1e9, "unit": "Gstreams/s", "cores": cores, "kind": "oracle",
                "sample": f"streams [0,{S}) of {n_streams} seeded (oracle rng_create)", "seconds": dt}
    cfgs = {"C2_u32": (W.C2, "fill_u32"), "C2_f32": (W.C2, "fill_f32"), "C1_u32": (W.C1, "fill_u32"),
            "C1_f32": (W.C1, "fill_f32"), "C1big_u32": (W.C1_BIG, "fill_u32"), "C3fill_u32": (W.C3_FILL, "fill_u32"),
            "C3_draw": (W.C3, "draw_reduce"), "C4_fill": (W.C4_FILL, "fill_u32"), "C4_draw": (W.C4_DRAW, "draw_reduce"),
            "N1_philox7_u32": (W.N1_PHILOX7, "fill_u32"), "N1_lcg32_u32": (W.N1_LCG32, "fill_u32"),
            "N1_philox7_draw": (W.N1_PHILOX7_DRAW, "draw_reduce"), "N1_philox10_draw": (W.N1_PHILOX10_DRAW, "draw_reduce"),
            "N1_lcg32_draw": (W.N1_LCG32_DRAW, "draw_reduce"), "N1_lcg64_draw": (W.N1_LCG64_DRAW, "draw_reduce"),
            "N1_lcg64both_draw": (W.N1_LCG64BOTH_DRAW, "draw_reduce"), "N3_mwc_draw": (W.N3_MWC_DRAW, "draw_reduce"), "N1_lcg64both_u32": (W.N1_LCG64BOTH, "fill_u32"),
            "N4_lfib521_f32": (W.N4_LFIB521, "fill_f32"), "N4_lfib1279_f32": (W.N4_LFIB1279, "fill_f32"),
            "N4_lfib521_draw": (W.N4_LFIB521_DRAW, "draw_reduce"), "N4_lfib1279_draw": (W.N4_LFIB1279_DRAW, "draw_reduce")}
    cfg, call = cfgs[workload]
    n = cfg.n_per_stream
    # calibrate on a small slice of the streams, then time one slice of about target_s
    gran = 256  # whole instances of every kind (xs1024: 32 streams, lagged Fibonacci: 256)
    S_probe = max(gran, min(cfg.n_streams, (1 << 22) // max(n, 1)) // gran * gran)
    r = oracle.Rng(cfg.kind, S_probe, cfg.seed)
    t0 = time.perf_counter()
    getattr(r, call)(n)
    dt = max(time.perf_counter() - t0, 1e-6)
    rate = S_probe * n / dt
    S = int(min(cfg.n_streams, max(S_probe, rate * target_s / n))) // gran * gran
    S = max(S, gran)
    r = oracle.Rng(cfg.kind, S, cfg.seed)
    t0 = time.perf_counter()
    getattr(r, call)(n)
    dt = time.perf_counter() - t0
    return {"value": S * n / dt / 1e9, "unit": "Gnum/s", "cores": cores, "kind": "oracle",
            "sample": f"streams [0,{S}) of {cfg.n_streams}, {n} draws each ({call})", "seconds": dt}


def run_reference(args) -> dict:
    """--impl reference: the oracle IS the reference arm for this tier.  Each step is a
    bounded sample of the workload (sized so the run ends within a few minutes)."""
    per_step = max(0.5, min(4.0, 120.0 / max(args.steps + args.warmup, 1)))
    for _ in range(args.warmup):
        oracle_sample_rate(args.workload, per_step)
    vals, last = [], None
    t0 = time.perf_counter()
    for _ in range(args.steps):
        last = oracle_sample_rate(args.workload, per_step)
        vals.append(last["value"])
    wall = time.perf_counter() - t0
    v = sum(vals) / len(vals)
    unit = last["unit"]
    return {"impl": "reference", "metric": METRIC, "value": v, "unit": unit, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": wall / args.steps * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "u32", "data": "synthetic (seeded streams; no dataset on this path)",
            "config": {"workload": args.workload, "sample": last["sample"]},
            "cpu_baseline": {"value": v, "unit": unit, "cores": last["cores"], "kind": "oracle", "sample": last["sample"]},
            "e2e": {"value": v, "unit": unit, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}


def hbm_ceilings(buf) -> dict:
    """context for the hbm roofline, measured live with library calls (not product code):
    a pure-store pass (memset) and a copy (read+write) over the 4 GiB buffer"""
    import torch
    out = {}
    half = buf.numel() // 2
    for name, fn, nbytes in (("memset_write_gbs", lambda: buf.zero_(), 4.0 * buf.numel()),
                             ("copy_rw_gbs", lambda: buf[:half].copy_(buf[half:]), 4.0 * buf.numel())):
        for _ in range(3):
            fn()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(10):
            fn()
        e1.record()
        torch.cuda.synchronize()
        out[name] = nbytes * 10 / (e0.elapsed_time(e1) * 1e-3) / 1e9
    return out


def run_e2e(job: Job, steps: int, warmup: int, world: int) -> dict:
    """the same metric through the host-buffer C-ABI call: pinned host memory, copies
    inside the timed region, every step"""
    import torch
    dist = torch.distributed if world > 1 else None
    if isinstance(job, FillJob):
        cfg = job.cfg
        host = torch.empty(cfg.draws_per_call, dtype=torch.float32 if job.f32 else torch.int32, pin_memory=True)
        fn = job.rng.fill_f32_host if job.f32 else job.rng.fill_u32_host
        one = lambda: [fn(host.data_ptr(), cfg.n_per_stream) for _ in range(cfg.calls)]  # noqa: E731
        h2d, d2h = 0, 4 * cfg.draws_per_call * cfg.calls
        api = "rng_fill_f32_host" if job.f32 else "rng_fill_u32_host"
    elif isinstance(job, DrawJob):
        cfg = job.cfg
        host = torch.empty(2 * cfg.n_streams, dtype=torch.int32, pin_memory=True)
        one = lambda: job.rng.draw_reduce_host(host.data_ptr(), cfg.n_per_stream)  # noqa: E731
        h2d, d2h = 0, 8 * cfg.n_streams
        api = "rng_draw_reduce_host"
    else:
        cfg = job.cfg
        host = torch.empty(cfg.L * cfg.L, dtype=torch.int8, pin_memory=True)
        host.copy_(job.spins)
        one = lambda: job.rng.ising_sweep_host(host.data_ptr(), cfg.L, cfg.beta, job.sweeps)  # noqa: E731
        h2d = d2h = cfg.L * cfg.L
        api = "ising_sweep_host"
    for _ in range(warmup):
        one()
    torch.cuda.synchronize()
    if dist:
        dist.barrier()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record()
    t0 = time.perf_counter()
    for _ in range(steps):
        one()
    ev1.record()
    torch.cuda.synchronize()
    wall_ms = (time.perf_counter() - t0) * 1e3
    ms = max(ev0.elapsed_time(ev1), wall_ms)  # the host call blocks: wall clock is the honest one
    if dist:
        ms = max_over_ranks(ms)
    val = job.units_per_step() * steps * world / (ms * 1e-3) / 1e9
    return {"value": val, "unit": job.unit, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h, "steps": steps,
            "ms_per_step": ms / steps, "api": api,
            "note": "inputs are scalars (kind, n_streams, seed); the result crosses the bus every step"
            if h2d == 0 else "lattice copied host->device and back every step"}


def run_fig1(kinds=("lcg32", "lcg64", "xorwow", "philox4x32_10", "xs1024w", "lfib521"), n=4096, step=37, max_blocks=148 * 16):
    """The analogue of the paper's Fig. 1: time per random number consumed in-register
    (rng_draw_reduce, n draws per stream) as a function of the number of 256-stream blocks, which the paper
    shows as a zig-zag commensurate with its 15 multiprocessors.  Returns {kind: [[blocks, ps_per_number], ...]}."""
    import torch
    import paper_1204_6193_b200 as pkg
    by_name = {v: k for k, v in pkg.KIND_NAMES.items()}
    out = {}
    red = torch.empty(2 * 256 * max_blocks, dtype=torch.int32, device="cuda")
    for name in kinds:
        rows = []
        for nb in range(step, max_blocks + 1, step):
            S = 256 * nb
            g = pkg.Rng(by_name[name], S, W.MASTER_SEED)
            g.draw_reduce(red, n)
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for _ in range(3):
                g.draw_reduce(red, n)
            e1.record()
            torch.cuda.synchronize()
            g.close()
            rows.append([nb, round(e0.elapsed_time(e1) / 3 * 1e9 / (S * n), 4)])  # picoseconds per number
        out[name] = rows
        best = min(r[1] for r in rows)
        log(f"[fig1] {name}: best {best:.3f} ps per number = {1e3 / best:.0f} Gnum/s at "
            f"{[r[0] for r in rows if r[1] == best][0]} blocks of 256 streams; "
            + " ".join(f"{r[0]}:{r[1]:.2f}" for r in rows[:: max(1, len(rows) // 16)]))
    return out


SHORT_DESC = {
    "C2_u32": "Philox4x32-10, 2^20 streams x 1024 u32 = 4 GiB per step (BASELINE configs[1])",
    "C2_f32": "Philox4x32-10, 2^20 streams x 1024 f32 = 4 GiB per step (BASELINE configs[1], float variant)",
}

# BASELINE.json's own configs besides the headline: (workload, steps, warmup) of --suite baseline
# plus row a1 (seeding) and the 4 GiB LCG64 supplement SURVEY.md 8(d) asks for beside C1
BASELINE_SUITE = [("C2_f32", 20, 3), ("C1_u32", 1000, 20), ("C1_f32", 1000, 20), ("C1big_u32", 20, 3), ("C3_draw", 20, 3),
                  ("C4_fill", 3, 1), ("C4_draw", 1, 1), ("C5b_philox", 1, 1), ("C5b_xorwow", 1, 1),
                  ("N2_seed_xs1024_random", 5, 3), ("N2_seed_xs1024_skip", 5, 3)]


def build_line(res: dict, args, world: int, cfg_info: dict, e2e=None, cpu=None, ceil=None, configs=None, sustained=None) -> dict:
    """the ONE stdout JSON object of the b200 arm (kept compact: the driver reads the last few KB of stdout).
    `res` is run_job()'s result for the headline workload, `configs` the other workloads' results."""
    line = {
        "metric": METRIC, "value": res["value"], "unit": res["unit"], "n_gpus": world, "steps": res["steps"],
        "warmup": res["warmup"], "ms_per_step": res["ms_per_step"], "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None,  # BASELINE.md holds no published number for this metric on this workload
        "dtype": res["dtype"], "data": "synthetic (seeded streams; this path has no dataset)", "impl": "b200",
        "config": {"workload": args.workload, "name": res["name"], **cfg_info, "parallelism": f"streams x{world}"},
        "clocks": res.get("clocks"), "gpu_launches": res["gpu_launches"], "roofline": res["roofline"],
    }
    if "paper_gtx480" in res:
        pg = res["paper_gtx480"]
        line["paper_gtx480"] = {"value": pg["value"], "unit": pg["unit"], "cite": pg["cite"], "ratio": round(pg["ratio"], 1)}
    if e2e:
        line["e2e"] = e2e
    if cpu:
        line["cpu_baseline"] = cpu
    if sustained:
        line["sustained"] = sustained
    if ceil:
        line["hbm_ceilings_measured_live"] = {k: round(v, 1) for k, v in ceil.items()}
    # only BASELINE.json's own configs ride on the line; --suite full's other workloads go to stderr / --dump
    own = {n for n, _, _ in BASELINE_SUITE}
    sig = lambda v: None if v is None else float(f"{v:.4g}")  # noqa: E731
    rows = [[c["workload"], round(c["value"], 2), c["unit"], c["roofline"]["bound"], c["roofline"]["frac"],
             c["roofline"].get("frac_vs_store_ceiling"), sig((c.get("cpu") or {}).get("value"))]
            for c in (configs or []) if c["workload"] in own]
    if rows:
        # roofline_frac: hbm rows against the measured copy bandwidth (frac_vs_store: against the live memset
        # ceiling -- a fill only writes); alu rows: ncu issue-active fraction.  cpu_oracle: the oracle on all host
        # cores on a ~2 s sample of the same workload, same unit
        line["configs_cols"] = ["workload", "value", "unit", "roofline_bound", "roofline_frac", "frac_vs_store", "cpu_oracle"]
        line["configs"] = rows
    return line


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--workload", default="C2_u32")
    ap.add_argument("--suite", default=None, choices=["primary", "baseline", "full"])
    ap.add_argument("--ising-sweeps", type=int, default=1000, help="sweeps per Ising step (config: 1000)")
    ap.add_argument("--e2e-steps", type=int, default=3)
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--sustained-s", type=float, default=2.0,
                    help="also run the headline step back to back for at least this many seconds (0 = skip)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--variant", default=None, help="NAME=VALUE: time a non-default kernel variant of the headline "
                    "workload (rng_set_variant, the library's test and measurement interface), e.g. xs1024=33")
    ap.add_argument("--dump", default=None, help="also write every workload's full result as a JSON list to this file")
    ap.add_argument("--dist-backend", default="nccl", choices=["nccl", "gloo"],
                    help="torch.distributed backend for N > 1 (nccl: one rank per GPU; gloo only for flow tests)")
    ap.add_argument("--fig1", action="store_true", help="instead of the benchmark: the paper's Fig. 1 on this GPU "
                    "(time per in-register random number against the number of 256-stream blocks); JSON on stdout")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "b200":
        log("[bench] note: timing rules ask for >= 3 warm-up steps")
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))

    if args.impl == "reference":
        if rank == 0:
            print(json.dumps(run_reference(args)), flush=True)
        return 0

    import torch
    import paper_1204_6193_b200 as pkg
    from paper_1204_6193_b200 import build as pkg_build
    if rank == 0:
        pkg_build.build()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    dev_index = local_rank % torch.cuda.device_count()  # == local_rank with one rank per GPU
    torch.cuda.set_device(dev_index)
    if world > 1:
        if args.dist_backend == "nccl":
            torch.distributed.init_process_group("nccl", device_id=torch.device("cuda", dev_index))
        else:  # gloo: only to exercise the N > 1 flow where ranks must share a GPU (tests); timings mean nothing
            torch.distributed.init_process_group(args.dist_backend)
        torch.distributed.barrier()
    pkg.lib()
    if args.fig1:
        if rank == 0:
            print(json.dumps({"fig1": run_fig1(), "unit": "ps per number", "x": "blocks of 256 streams, 4096 draws per stream",
                              "cite": "PAPER.md:52"}), flush=True)
        return 0
    suite = args.suite or ("baseline" if world == 1 and args.workload == "C2_u32" else "primary")
    buf = torch.empty(1 << 30, dtype=torch.int32, device="cuda")  # 4 GiB, reused by every workload (> L2)

    # write-only and copy ceilings of this box, measured before the timed region with library calls
    ceil = hbm_ceilings(buf)
    store_gbs = ceil["memset_write_gbs"]

    job = make_job(args.workload, rank, world, buf, args.ising_sweeps)
    variant = None
    if args.variant:  # measurements of the non-default kernel variants (bit-identical)
        vn, vv = args.variant.split("=")
        job.rng.set_variant(vn, int(vv))
        variant = {vn: int(vv)}
    res = run_job(job, args.steps, args.warmup, world, sample_clocks=True, dev_index=dev_index, store_gbs=store_gbs)
    sustained = None
    if world == 1 and args.sustained_s > 0 and not isinstance(job, (IsingJob, SeedJob)):
        # the same step back to back for at least --sustained-s seconds: the power-limited regime beside the burst
        n_sus = max(args.steps, int(args.sustained_s * 1e3 / max(res["ms_per_step"], 1e-3)) + 1)
        rs = run_job(job, n_sus, 0, world, sample_clocks=True, dev_index=dev_index, store_gbs=store_gbs)
        sustained = {"value": round(rs["value"], 2), "unit": rs["unit"], "steps": n_sus, "ms_per_step": round(rs["ms_per_step"], 5),
                     "seconds": round(rs["ms_per_step"] * n_sus / 1e3, 2), "roofline_frac": rs["roofline"]["frac"],
                     "frac_vs_store_ceiling": rs["roofline"].get("frac_vs_store_ceiling"), "clocks": rs.get("clocks")}
        log(f"[bench] sustained {args.workload}: {rs['value']:.2f} {rs['unit']} over {sustained['seconds']} s, clocks {rs.get('clocks')}")
    e2e = None if args.no_e2e else run_e2e(job, args.e2e_steps, 1, world)
    cfg_info = {"desc": SHORT_DESC.get(args.workload, res["name"]),
                "streams_per_gpu": getattr(getattr(job, "cfg", None), "n_streams", getattr(job, "n_local", None)),
                "l2": "64 MiB lattice is L2-resident by design (DESIGN.md s7)" if isinstance(job, IsingJob)
                else "4 GiB output per step > 126 MB L2, no flush needed"}
    if variant:
        cfg_info["variant"] = variant
    job.close()
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        cpu = oracle_sample_rate(args.workload, 8.0)
        cpu["seconds"] = round(cpu["seconds"], 2)
        one = oracle_sample_rate(args.workload, 6.0, threads=1)
        cpu["single_thread"] = {"value": one["value"], "unit": one["unit"], "cores": 1, "sample": one["sample"],
                                "seconds": round(one["seconds"], 2)}

    configs = []
    todo = BASELINE_SUITE if suite == "baseline" else SUITE if suite == "full" else []
    for name, k, w in todo:
        if name == args.workload:
            continue
        j = make_job(name, rank, world, buf, args.ising_sweeps)
        r = run_job(j, k, w, world, sample_clocks=False, dev_index=dev_index, store_gbs=store_gbs)
        j.close()
        r["workload"] = name
        if rank == 0 and world == 1 and not args.no_cpu_baseline and suite == "baseline":
            r["cpu"] = oracle_sample_rate(name, 2.0)
        configs.append(r)
        rl = r["roofline"]
        extra = f" (vs store ceiling {rl['frac_vs_store_ceiling']:.3f})" if "frac_vs_store_ceiling" in rl else \
            f" (ncu issue {rl.get('ncu_issue_active_pct')}%, {rl.get('ncu_binding_pipe')})" if rl["bound"] == "alu" else ""
        log(f"[bench] {name} = {r['name']}: {r['value']:.2f} {r['unit']}  {r['ms_per_step']:.3f} ms/step  "
            f"roofline {rl['bound']} {rl['frac']:.3f}{extra}")

    if rank == 0:
        line = build_line(res, args, world, cfg_info, e2e, cpu, ceil if world == 1 else None, configs, sustained)
        if args.dump:
            with open(args.dump, "w") as f:
                json.dump([dict(res, workload=args.workload)] + configs, f, indent=1)
        print(json.dumps(line), flush=True)
    if world > 1:
        torch.distributed.barrier()
        torch.distributed.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
