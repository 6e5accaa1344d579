#!/usr/bin/env python
"""bench.py -- AES-256-GCM encrypt GB/s on a 4 GiB message (BASELINE.json config 5), device-timed.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--size-mib M]

One "step" = one pass of the whole hot path (counters, AES rounds, payload
XOR, GHASH fold + combine, tag) over one 4 GiB synthetic message that is already resident in HBM.
Prints ONE JSON line (rank 0).  With N > 1 (torchrun) every rank encrypts its own message on its
own GPU: messages are independent, there is no data-path collective ("scaling": "weak"); NCCL is
used only for the barrier and the max-over-ranks of the device time.

  value      payload GB/s (1e9 bytes), all ranks' bytes / max-over-ranks device time of the K steps
  e2e        same metric through gcm_encrypt_host(): pinned HOST buffers in and out, the H2D and D2H
             copies inside the timed region
  roofline   achieved payload GB/s of the fused kernel vs the shared-memory-pipe bound derived in
             DESIGN.md section 6 (the binding unit; the HBM figure is reported beside it)
  cpu_baseline  the CPU oracle, as it stands, on the host cores, on a bounded sample of the workload

--impl reference times the oracle itself (this tier has no reference implementation to install).
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import tempfile
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "AES-256-GCM encrypt GB/s (device-timed, 4 GiB msg)"
UNIT = "GB/s"
WORKLOAD = "C5: AES-256-GCM encrypt, one 4 GiB uniform-random message, 2880-byte FITS header AAD, 96-bit IV"


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--size-mib", type=float, default=4096.0, help="payload MiB (default: the 4 GiB of config 5)")
    ap.add_argument("--e2e-steps", type=int, default=3)
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-supplementary", action="store_true", help="leave the other configs out of the default line")
    ap.add_argument("--cpu-sample-mib", type=float, default=384.0)
    ap.add_argument("--workload", default="c5",
                    choices=["c5", "c5-decrypt", "c5-ghash", "c5-aes128", "c5-tensor", "c5-aes128-tensor", "c2", "c3", "c4", "latency", "frame", "datasum", "phases", "sizes"],
                    help="c5 = the headline (default); the others are the supplementary measurements of DESIGN.md section 10")
    return ap.parse_args()


# ---------------------------------------------------------------------------------------------------
# clocks during the timed region (B200_PROFILING.md recipe)
# ---------------------------------------------------------------------------------------------------
class ClockSampler:
    QUERY = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
             "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
             "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.proc = None
        self.path = None

    def start(self):
        try:
            fd, self.path = tempfile.mkstemp(prefix="clocks_", suffix=".csv")
            os.close(fd)
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.QUERY, "--format=csv,noheader,nounits",
                 "-lms", "100"], stdout=open(self.path, "w"), stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self) -> dict:
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.proc is None:
            return out
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, reasons, power = [], [], set(), []
        try:
            for line in open(self.path):
                f = [x.strip() for x in line.split(",")]
                if len(f) < 9:
                    continue
                try:
                    sm.append(float(f[1])); mx.append(float(f[2])); power.append(float(f[3]))
                except ValueError:
                    continue
                for name, val in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[5:9]):
                    if val.lower().startswith("active"):
                        reasons.add(name)
            os.unlink(self.path)
        except Exception:
            pass
        if sm:
            # samples under load: the upper half (idle samples before/after the region sit at low clocks)
            load = sorted(sm)[len(sm) // 2:]
            out.update(sm_mhz=statistics.median(load), sm_max_mhz=max(mx), reasons=sorted(reasons),
                       samples=len(sm), power_w_max=max(power) if power else None)
        return out


# ---------------------------------------------------------------------------------------------------
# roofline
# ---------------------------------------------------------------------------------------------------
def measured_peaks() -> dict:
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        d["_source"] = "measured"
        return d
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0, "_source": "fallback"}


MIX_FILE = os.path.join(ROOT, "profiles", "sass_mix.json")


def load_mix(key: str) -> dict:
    """Executed instruction mix of a kernel's row loop per warp-row (32 blocks), written by
    `python -m paper_2602_23067_b200.profile_tools mix` from the ncu source page of the shipped kernel
    (profiles/README_r02.md has the commands).  The roofline is built from it, not from a typed-in formula."""
    try:
        return json.load(open(MIX_FILE))[key]
    except Exception as e:
        raise SystemExit("bench.py: %s has no usable entry %r (%s): capture it as profiles/README_r02.md says; the roofline "
                         "is derived from the shipped binary's executed mix and is not guessed" % (MIX_FILE, key, e))


def mix_matches_library(key: str):
    """True / False: the mix entry was captured from the very library file that is loaded now (size and SHA-256 stored
    by profile_tools mix); None when the entry predates that record."""
    import hashlib
    fp = load_mix(key).get("library")
    if not fp:
        return None
    import paper_2602_23067_b200 as G
    data = open(G.library_path(), "rb").read()
    return fp.get("bytes") == len(data) and fp.get("sha256") == hashlib.sha256(data).hexdigest()


def pipe_bound_gbs(key: str, nr: int, sm_count: int, sm_mhz: float, rates: dict = None, ghash_only: bool = False) -> dict:
    """Shared-memory-pipe (LSU data pipe) bound.  An SM retires one 128-byte shared-memory wavefront per cycle: a
    conflict-free LDS.32 of a warp is one wavefront, an LDS.64 two, an LDS.128 four; a warp-row is 32 blocks, one per
    lane, so wavefronts per warp-row = bank-lanes per block and cycles per block per SM = that / 32.
      lanes            from the kernel's own executed mix (load_mix): the binding roofline north_star defines
      with measured rates   the same counts against gcm_measure_pipe_rates' LDS.32 / LDS.128 rates of this device
      yardsticks       kernel-independent ('so a bloated kernel cannot flatter itself'): the plain
                       table design (16 T-table reads per round + a 16-lookup 8-bit Shoup multiply: 16 nr + 64 lanes)
                       and the AES table reads alone with every hoistable read hoisted (16 nr - 27 + 15/8)."""
    e = load_mix(key)["per_warp_row"]
    lanes = e["lds32"] + 2.0 * e["lds64"] + 4.0 * e["lds128"] + 4.0 * e.get("sts128", 0.0)
    if key.startswith("tc2_"):
        # AES warps + tensor-core GHASH: the tensor core reads its B operand (the bit matrices) from shared memory through the
        # same data pipe; those wavefronts belong to no instruction, so the launch's measured total is the count that binds
        lanes = max(lanes, e.get("shared_wavefronts_total", 0.0))
    glob = 4.0 * (e["ldg128"] + e["stg128"])
    scale = sm_count * sm_mhz * 1e6 * 16.0 / 1e9
    out = {"mix": key, "lanes_per_block": lanes, "global_lanes_per_block": glob, "cycles_per_block_per_sm": lanes / 32.0,
           "gbs": scale / (lanes / 32.0), "gbs_with_global_wavefronts": scale / ((lanes + glob) / 32.0),
           "counts_per_block": {k: round(e.get(k, 0.0), 3) for k in ("lds32", "lds64", "lds128", "sts128", "ldg128", "stg128", "shared_wavefronts_total")},
           "alu_thread_instructions_per_block": e["by_pipe_warp_instructions"].get("alu"),
           "fma_thread_instructions_per_block": e["by_pipe_warp_instructions"].get("fma"),
           "thread_instructions_per_block": e["warp_instructions"]}
    if rates and rates.get("lds32") and rates.get("lds128"):
        cyc = e["lds32"] / rates["lds32"] + 2.0 * e["lds64"] / (2.0 * rates["lds128"]) + e["lds128"] / rates["lds128"]
        if key.startswith("tc2_"):
            cyc = lanes / rates["lds32"]          # every wavefront of the launch at the measured wavefront rate
        out["gbs_measured_rates"] = scale / cyc
    naive = 64.0 if ghash_only else 16.0 * nr + 64.0
    out["yardsticks"] = {"plain_table_design_lanes": naive, "plain_table_design_gbs": scale / (naive / 32.0)}
    if not ghash_only:
        floor = 16.0 * nr - 27.0 + 15.0 / 8.0
        out["yardsticks"].update(aes_reads_only_lanes=floor, aes_reads_only_gbs=scale / (floor / 32.0))
    return out


def roofline_dict(pb: dict, achieved: float, peaks: dict, hbm_bytes_per_byte: int) -> dict:
    """The contract's roofline object for a kernel bound by the shared-memory data pipe."""
    hbm_peak = float(peaks["hbm_gbs"])
    y = pb["yardsticks"]
    r = {"bound": "alu", "unit_pipe": "lsu_shared",
         "pipe": "shared-memory data pipe (LSU): %.1f bank-lanes per 16-byte block from the kernel's executed mix "
                 "(%s), 32 per SM-cycle" % (pb["lanes_per_block"], pb["mix"]),
         "achieved": achieved, "peak": pb["gbs"], "unit": UNIT, "frac": achieved / pb["gbs"],
         "frac_with_global_wavefronts": achieved / pb["gbs_with_global_wavefronts"],
         "counts_per_block": pb["counts_per_block"],
         "yardsticks": {k: (round(v, 1) if isinstance(v, float) else v) for k, v in y.items()},
         "frac_of_plain_table_design": achieved / y["plain_table_design_gbs"],
         "hbm": {"achieved": hbm_bytes_per_byte * achieved, "peak": hbm_peak, "unit": "GB/s",
                 "frac": hbm_bytes_per_byte * achieved / hbm_peak, "of": peaks["_source"]}}
    if "aes_reads_only_gbs" in y:
        r["frac_of_aes_reads_only_floor"] = achieved / y["aes_reads_only_gbs"]
    if "gbs_measured_rates" in pb:
        r["peak_measured_rates"] = pb["gbs_measured_rates"]
        r["frac_measured_rates"] = achieved / pb["gbs_measured_rates"]
    return r


def tensor_roofline(gbs: float, sm_count: int, sm_mhz: float, peaks: dict, rates: dict = None) -> dict:
    """Roofline of gcm_ghash_tc_kernel.  Work: one 128 x 128 bit matrix-vector product per 16-byte block = 2 x 16,384
    flop on e2m1 (fp4) operands.  `peak` follows the contract: the measured dense bf16 rate of MEASURED_PEAKS.json
    (cuBLAS, burst) x the nominal fp4 : bf16 ratio of 4 (9 / 2.25 PFLOP/s).  cuBLAS runs power-capped near 1.3 GHz,
    this kernel at the full SM clock, so the fraction can exceed 1; the tight bound is the instruction rate: a
    128 x 128 x 64 kind::mxf4 MMA takes 64 SM-cycles (measured with back-to-back MMAs on this device), i.e. one block
    per SM-cycle."""
    flop_per_byte = 2.0 * 128 * 128 / 16.0
    achieved = gbs * 1e9 * flop_per_byte / 1e12
    r = {"bound": "tensor", "unit": "TFLOP/s", "achieved": achieved, "dtype": "fp4 e2m1 (kind::mxf4), fp32 accumulate",
         "flop_per_payload_byte": flop_per_byte, "traffic": None}
    try:            # dram bytes of one launch from the committed ncu --set full capture, scaled by size
        t = json.load(open(os.path.join(ROOT, "profiles", "traffic.json")))["ghash_tc"]
        r["traffic_per_payload_byte"] = t["dram_bytes_per_payload_byte"]
    except Exception:
        pass
    bf16 = peaks.get("bf16_tflops")
    if bf16:
        r.update(peak=4.0 * float(bf16), frac=achieved / (4.0 * float(bf16)),
                 peak_how="bf16_tflops of MEASURED_PEAKS.json (%s) x 4 (nominal fp4 : bf16)" % peaks["_source"])
    else:
        r.update(peak=4.0 * 1590.0, frac=achieved / (4.0 * 1590.0), peak_how="fallback 1.59 PFLOP/s bf16 x 4 (of fallback)")
    blocks_per_cycle = float(rates["mma_mxf4_blocks"]) if rates and rates.get("mma_mxf4_blocks") else 1.0
    issue = sm_count * sm_mhz * 1e6 * 16.0 * blocks_per_cycle / 1e9      # GB/s at the measured MMA rate (nominal: one block per SM-cycle)
    r.update(mma_blocks_per_sm_cycle=blocks_per_cycle, peak_mma_issue_rate_gbs=issue, frac_of_mma_issue_rate=gbs / issue,
             hbm={"achieved": gbs, "peak": float(peaks["hbm_gbs"]), "unit": "GB/s", "frac": gbs / float(peaks["hbm_gbs"]),
                  "of": peaks["_source"]})
    return r


def step_with(ctx, aad, ct, stream, G):
    import torch
    d_s = torch.zeros(16, dtype=torch.uint8, device="cuda")
    return lambda: G.gcm_ghash_async(ctx, aad, ct, d_s, stream)


def traffic_per_launch(payload_bytes: int, key: str = None):
    """dram bytes per launch from the committed ncu --set full capture (profiles/), scaled by size."""
    p = os.path.join(ROOT, "profiles", "traffic.json")
    try:
        d = json.load(open(p))
        if key:
            d = d[key]
        return d["dram_bytes_per_payload_byte"] * payload_bytes
    except Exception:
        return None


# ---------------------------------------------------------------------------------------------------
# the CPU oracle legs (cpu_baseline of our arm, and the whole --impl reference arm)
# ---------------------------------------------------------------------------------------------------
def oracle_sample_gbs(sample_bytes: int):
    """AES-256-GCM encrypt of a `sample_bytes` prefix-sized message of the same recipe on the host
    cores: CTR chunked over all cores, GHASH the sequential Horner chain on one (oracle as it stands)."""
    import numpy as np
    from oracle import oracle as O
    import workloads
    cores = os.cpu_count() or 1
    m = workloads.config_c5(payload_bytes=sample_bytes)
    O.lib()
    t0 = time.perf_counter()
    ct, tag = O.gcm_encrypt_threaded(m.key, m.iv, m.aad, m.payload, threads=cores, segment_blocks=0)
    dt = time.perf_counter() - t0
    assert ct.size == sample_bytes and len(tag) == 16
    return sample_bytes / dt / 1e9, cores, dt


def cpu_context(key, iv):
    """Context figures beside the oracle baseline: the oracle on ONE thread, and the installed
    OpenSSL (AES-NI / VPCLMULQDQ) on one core and on all cores -- the kind of CPU baseline the paper's speed-up
    figures refer to.  Bounded samples; none of this is a target."""
    import numpy as np
    from concurrent.futures import ThreadPoolExecutor
    from oracle import oracle as O
    out = {}
    small = np.zeros(16 << 20, np.uint8)
    t0 = time.perf_counter()
    O.gcm_encrypt(key, iv, b"", small)
    out["oracle_1_thread_GBps"] = small.size / (time.perf_counter() - t0) / 1e9
    try:
        from cryptography.hazmat.primitives.ciphers.aead import AESGCM
        big = bytes(256 << 20)
        a = AESGCM(key)
        a.encrypt(iv, big[:1 << 20], b"")
        t0 = time.perf_counter()
        a.encrypt(iv, big, b"")
        out["openssl_1_core_GBps"] = len(big) / (time.perf_counter() - t0) / 1e9
        cores = os.cpu_count() or 1
        with ThreadPoolExecutor(cores) as ex:
            t0 = time.perf_counter()
            list(ex.map(lambda i: len(AESGCM(key).encrypt(iv, big, b"")), range(cores)))
            out["openssl_all_cores_GBps"] = cores * len(big) / (time.perf_counter() - t0) / 1e9
        out["openssl_cores"] = cores
        out["openssl_note"] = "one-shot AESGCM.encrypt of 256 MiB per call, output allocation included"
    except Exception as e:                      # context only
        out["openssl"] = "unavailable: %s" % type(e).__name__
    return out


def pcie_duplex_gbs(nbytes: int = 1 << 30, reps: int = 3) -> dict:
    """What the host link gives: one pinned H2D copy and one pinned D2H copy of `nbytes` each, alone and both at once
    on two streams (the e2e path moves the message both ways at the same time).  GB/s per direction, best of reps."""
    import torch
    h_a = torch.empty(nbytes, dtype=torch.uint8).pin_memory()
    h_b = torch.empty(nbytes, dtype=torch.uint8).pin_memory()
    d_a = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
    d_b = torch.zeros(nbytes, dtype=torch.uint8, device="cuda")
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()

    def run(h2d: bool, d2h: bool) -> float:
        best = 1e30
        for _ in range(reps + 1):
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            if h2d:
                with torch.cuda.stream(s1):
                    d_a.copy_(h_a, non_blocking=True)
            if d2h:
                with torch.cuda.stream(s2):
                    h_b.copy_(d_b, non_blocking=True)
            torch.cuda.synchronize()
            best = min(best, time.perf_counter() - t0)
        return nbytes / best / 1e9

    out = {"h2d_alone": run(True, False), "d2h_alone": run(False, True), "per_direction_duplex": run(True, True),
           "bytes": nbytes, "how": "torch copy_ of pinned buffers, one cudaMemcpyAsync per direction, host wall clock, best of %d" % reps}
    del h_a, h_b, d_a, d_b
    return out


def oracle_batch_gbs(msgs, what: str) -> dict:
    """cpu_baseline of the batched configs: the oracle as it stands, one whole message per task, tasks spread over the
    host cores (independent messages: SURVEY.md 8(d))."""
    from concurrent.futures import ThreadPoolExecutor
    from oracle import oracle as O
    cores = os.cpu_count() or 1
    O.lib()
    t0 = time.perf_counter()
    with ThreadPoolExecutor(cores) as ex:
        tags = list(ex.map(lambda m: O.gcm_encrypt(m.key, m.iv, m.aad, m.payload)[1], msgs))
    dt = time.perf_counter() - t0
    nbytes = sum(m.payload.size for m in msgs)
    assert len(tags) == len(msgs)
    return {"value": nbytes / dt / 1e9, "unit": UNIT, "cores": cores, "kind": "oracle", "seconds": dt,
            "sample": "%s: %d messages, %d bytes, one message per task over %d threads" % (what, len(msgs), nbytes, cores)}


def run_reference(args):
    """--impl reference: the oracle, as it stands, on the host cores; each step a bounded sample."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    sample = int(min(args.cpu_sample_mib, 16.0) * (1 << 20))
    steps, warm = max(1, min(args.steps, 5)), max(0, min(args.warmup, 1))
    for _ in range(warm):
        oracle_sample_gbs(sample)
    t0 = time.perf_counter()
    cores = 1
    for _ in range(steps):
        _, cores, _ = oracle_sample_gbs(sample)
    dt = time.perf_counter() - t0
    gbs = steps * sample / dt / 1e9
    sample_txt = "first %.0f MiB-sized message of the C5 recipe per step (the 4 GiB message would take minutes)" % (sample / 2 ** 20)
    line = {
        "impl": "reference", "metric": METRIC, "value": gbs, "unit": UNIT, "n_gpus": args.gpus,
        "steps": steps, "warmup": warm, "ms_per_step": dt / steps * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "u8", "data": "synthetic",
        "config": {"workload": WORKLOAD, "sample": sample_txt},
        "cpu_baseline": {"value": gbs, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample_txt},
        "e2e": {"value": gbs, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


# ---------------------------------------------------------------------------------------------------
# our arm
# ---------------------------------------------------------------------------------------------------
def run_ours(args):
    import numpy as np
    import torch
    import torch.distributed as dist
    import paper_2602_23067_b200 as G
    import workloads

    from paper_2602_23067_b200 import replicas
    rank, local, world = replicas.rank_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local)
    G.gcm_set_device(local)
    replicas.init("nccl", torch.device("cuda", local))
    barrier = replicas.barrier

    n = int(args.size_mib * (1 << 20))
    m = workloads.config_c5(payload_bytes=n, with_payload=False)
    key = replicas.replica_key(m.key, rank)                      # one independent message per rank
    gen = torch.Generator(device="cuda")
    gen.manual_seed(replicas.replica_seed(workloads.SEEDS["C5"], rank))
    # uniform random bytes, generated on the device 8 bytes at a time
    pt = torch.randint(-2 ** 63, 2 ** 63 - 1, ((n + 7) // 8,), dtype=torch.int64, device="cuda", generator=gen).view(torch.uint8)[:n]
    ct = torch.empty(n, dtype=torch.uint8, device="cuda")
    aad = torch.from_numpy(m.aad).cuda()
    d_tag = torch.zeros(16, dtype=torch.uint8, device="cuda")
    ctx = G.gcm_init(key)
    stream = torch.cuda.current_stream()
    # a1 + a2 (key schedule, H, power and multiplier tables) reported separately: a second context
    # built on a warm library, device time of the setup kernel and host wall clock of the whole gcm_init
    torch.cuda.synchronize()
    es0, es1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t_s = time.perf_counter()
    es0.record()
    ctx2 = G.gcm_init(key)
    es1.record()
    torch.cuda.synchronize()
    setup = {"gcm_init_wall_ms": (time.perf_counter() - t_s) * 1e3, "setup_device_ms": es0.elapsed_time(es1)}
    G.gcm_destroy(ctx2)
    rates = G.gcm_measure_pipe_rates() if rank == 0 else {}   # unit rates behind the roofline (outside the timed region)

    def step():
        G.gcm_encrypt_async(ctx, m.iv, aad, pt, ct, d_tag, stream)

    for _ in range(max(3, args.warmup)):
        step()
    torch.cuda.synchronize()

    # blocks sampled for the parity check of the cpu_baseline leg (the oracle itself is only touched there)
    samples = []
    if rank == 0:
        rs = np.random.default_rng(5)
        nblk = n // 16
        for g in sorted({0, nblk - 1, *rs.integers(0, max(1, nblk), 6).tolist()}):
            samples.append((int(g), ct[16 * g: 16 * g + 16].cpu().numpy() ^ pt[16 * g: 16 * g + 16].cpu().numpy()))

    sampler = ClockSampler(local)
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps + 1)]
    barrier()
    torch.cuda.synchronize()
    if rank == 0:
        sampler.start()
    ev[0].record(stream)
    for i in range(args.steps):
        step()
        ev[i + 1].record(stream)
    torch.cuda.synchronize()
    barrier()
    clocks = sampler.stop() if rank == 0 else {}
    total_ms = ev[0].elapsed_time(ev[-1])
    per = [ev[i].elapsed_time(ev[i + 1]) for i in range(args.steps)]
    total_ms = replicas.max_over_ranks(total_ms, "cuda")
    value = replicas.aggregate_gbs(n, args.steps, total_ms, world)

    # end to end: pinned host buffers through gcm_encrypt_host (H2D + kernels + D2H inside the region)
    e2e = None
    if not args.no_e2e:
        h_pt = torch.empty(n, dtype=torch.uint8).pin_memory()
        h_ct = torch.empty(n, dtype=torch.uint8).pin_memory()
        h_pt.copy_(pt)
        h_aad = m.aad
        G.gcm_encrypt_host(ctx, m.iv, h_aad, h_pt, h_ct, stream)          # warm-up (allocates staging)
        barrier()
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for _ in range(args.e2e_steps):
            tag_h = G.gcm_encrypt_host(ctx, m.iv, h_aad, h_pt, h_ct, stream)
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        dt = replicas.max_over_ranks(dt, "cuda")
        assert tag_h == d_tag.cpu().numpy().tobytes(), "host-path tag differs from device-path tag"
        assert torch.equal(h_ct[:4096], ct[:4096].cpu()) and torch.equal(h_ct[-4096:], ct[-4096:].cpu())
        e2e = {"value": replicas.aggregate_gbs(n, args.e2e_steps, dt * 1e3, world), "unit": UNIT,
               "h2d_bytes_per_step": n + int(m.aad.size), "d2h_bytes_per_step": n + 16,
               "steps": args.e2e_steps, "how": "gcm_encrypt_host: pinned host in/out, chunked H2D -> fused kernel -> D2H"}
        del h_pt, h_ct
        if rank == 0:
            # the bound of this leg: the message crosses the host link once in each direction, at the same time
            link = pcie_duplex_gbs(min(n, 1 << 30))
            e2e["pcie_peak"] = link["per_direction_duplex"]
            e2e["frac"] = e2e["value"] / world / link["per_direction_duplex"]
            e2e["pcie"] = link

    # the SM clock the dominant kernel really ran at in the last timed step, from the kernel's own clock64 / %globaltimer
    kernel_clock = None
    if rank == 0 and n >= G.TC2_AUTO_BYTES[256]:
        try:
            mhz, k_ms = G.gcm_debug_tc2_clock(ctx)
            kernel_clock = {"sm_mhz": mhz, "kernel_ms": k_ms}
        except G.GcmError:
            kernel_clock = None

    # the shared-memory table kernel on the same message, beside it (not the reported value)
    table_engine = None
    if rank == 0 and n >= G.TC2_AUTO_BYTES[256]:
        G.gcm_set_ghash_engine(ctx, G.GCM_GHASH_TABLE)
        for _ in range(3):
            step()
        torch.cuda.synchronize()
        t0e, t1e = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        t0e.record()
        for _ in range(args.steps):
            step()
        t1e.record()
        torch.cuda.synchronize()
        tab_ms = t0e.elapsed_time(t1e) / args.steps
        tab_gbs = n / (tab_ms * 1e-3) / 1e9
        tpb = pipe_bound_gbs("fused_aes256_enc", 14, torch.cuda.get_device_properties(local).multi_processor_count,
                             float(measured_peaks().get("sm_max_mhz", 1965.0)), rates)
        table_engine = {"kernel": "gcm_fused_kernel<14, ENCRYPT, 512> (GCM_GHASH_TABLE)", "value": tab_gbs, "unit": UNIT, "ms_per_step": tab_ms,
                        "peak": tpb["gbs"], "frac": tab_gbs / tpb["gbs"], "lanes_per_block": tpb["lanes_per_block"]}
        G.gcm_set_ghash_engine(ctx, G.GCM_GHASH_AUTO)
    G.gcm_destroy(ctx)
    if rank != 0:
        replicas.finish()
        return

    peaks = measured_peaks()
    sm_count = torch.cuda.get_device_properties(local).multi_processor_count
    kernel_ms = statistics.mean(per)
    achieved = n / (kernel_ms * 1e-3) / 1e9
    sm_mhz = float(peaks.get("sm_max_mhz", 1965.0))
    # Under the default engine an aligned message of 384 MiB and more (T2_AUTO_BYTES_256) runs as three chained launches: the row kernel over
    # the AAD and the first 254 blocks, gcm_tc2_kernel (AES warps + tensor-core GHASH warps) over the whole 128-block
    # slices, the row kernel over the rest and the length block.  The dominant kernel is gcm_tc2_kernel (99.8 % of a step's
    # device time in profiles/launches_r02_c5.csv); kernel_ms is the step (its two short links included).
    uses_tc2 = n >= G.TC2_AUTO_BYTES[256]
    mix_key = "tc2_aes256_enc" if uses_tc2 else "fused_aes256_enc"
    pb = pipe_bound_gbs(mix_key, 14, sm_count, sm_mhz, rates)
    roofline = roofline_dict(pb, achieved, peaks, 2)
    roofline.update({
        "peak_source": "derived (DESIGN.md section 6): %d SMs x %.0f MHz (MEASURED_PEAKS sm_max_mhz, %s) x 16 B / %.3f cycles; "
                       "lanes from %s" % (sm_count, sm_mhz, peaks["_source"], pb["cycles_per_block_per_sm"], os.path.relpath(MIX_FILE, ROOT)),
        "traffic": traffic_per_launch(n, "tc2" if uses_tc2 else None),
        "algorithmic_bytes_per_launch": 2 * n,
        "rates": {"unit": "thread-operations per SM-cycle, measured by gcm_measure_pipe_rates on this device",
                  **{k: round(v, 2) for k, v in rates.items()}},
        "kernel": "gcm_tc2_kernel<14, ENCRYPT> (+ two short gcm_fused_kernel links)" if uses_tc2 else "gcm_fused_kernel<14, ENCRYPT, 512>",
        "kernel_ms_mean": kernel_ms,
        "kernel_ms_median": statistics.median(per),
        "mix_captured_from_loaded_library": mix_matches_library(mix_key),
    })
    if clocks.get("sm_mhz"):
        roofline["frac_at_sampled_clock"] = achieved / pipe_bound_gbs(mix_key, 14, sm_count, clocks["sm_mhz"])["gbs"]
    if uses_tc2:
        # gcm_tc2_kernel's own wavefront total includes its hand-over stores and the tensor core's operand reads, so an
        # extra wavefront in the kernel would lower that peak and raise the fraction.  The headline `peak` / `frac` are
        # therefore held against the kernel-independent floor (the AES table reads alone, every hoistable read hoisted:
        # 16 nr - 27 + 15/8 lanes per block); the kernel's own count stays beside it as *_self_derived.
        y = pb["yardsticks"]
        roofline["peak_self_derived"], roofline["frac_self_derived"] = roofline["peak"], roofline["frac"]
        roofline["peak"], roofline["frac"] = y["aes_reads_only_gbs"], achieved / y["aes_reads_only_gbs"]
        roofline["peak_source"] = ("kernel-independent: AES table reads only, %.2f lanes per 16-byte block (16 x 14 - 27 + 15/8), 32 per SM-cycle, "
                                   "%d SMs x %.0f MHz (MEASURED_PEAKS sm_max_mhz, %s); peak_self_derived: the %.1f wavefront-lanes per block "
                                   "measured for this kernel (%s)" % (y["aes_reads_only_lanes"], sm_count, sm_mhz, peaks["_source"],
                                                                    pb["lanes_per_block"], os.path.relpath(MIX_FILE, ROOT)))
        if clocks.get("sm_mhz"):
            roofline["frac_self_derived_at_sampled_clock"] = roofline["frac_at_sampled_clock"]
            roofline["frac_at_sampled_clock"] = roofline["frac"] * sm_mhz / clocks["sm_mhz"]
        if kernel_clock:
            # nvidia-smi (clocks.sm_mhz) keeps showing the maximum while a tcgen05 kernel runs below it: the kernel's own
            # cycle and nanosecond counters (gcm_debug_tc2_clock, CTA 0 of the last timed step) give the clock that applies
            roofline["sm_mhz_kernel"] = kernel_clock["sm_mhz"]
            roofline["kernel_ms_by_globaltimer"] = kernel_clock["kernel_ms"]
            roofline["frac_at_kernel_clock"] = roofline["frac"] * sm_mhz / kernel_clock["sm_mhz"]
            roofline["frac_self_derived_at_kernel_clock"] = roofline["frac_self_derived"] * sm_mhz / kernel_clock["sm_mhz"]
            roofline["frac_at_sampled_clock"] = roofline["frac_at_kernel_clock"]
            roofline["sampled_clock_note"] = ("frac_at_sampled_clock uses sm_mhz_kernel (measured inside the kernel); nvidia-smi sampled %s MHz"
                                              % clocks.get("sm_mhz"))
        roofline["pipe"] = ("shared-memory data pipe (LSU): %.1f wavefront-lanes per 16-byte block measured for the launch (%s): AES table reads, "
                            "the hand-over of the ciphertext to the GHASH warps, and the tensor core's reads of the bit matrices; 32 per SM-cycle. "
                            "GHASH itself runs on tcgen05.mma kind::mxf4" % (pb["lanes_per_block"], pb["mix"]))
        roofline["tensor_pipe"] = {"blocks_per_sm_cycle_peak": rates.get("mma_mxf4_blocks"), "note": "one GHASH block per SM-cycle available; the kernel needs 8/7 MMA-blocks per block at the AES rate: about 14 % of the pipe"}
        roofline["table_engine"] = table_engine

    cpu = None
    verified = 0
    if not args.no_cpu_baseline:
        sample = int(args.cpu_sample_mib * (1 << 20))
        gbs, cores, dt = oracle_sample_gbs(sample)
        cpu = {"value": gbs, "unit": UNIT, "cores": cores, "kind": "oracle", "seconds": dt,
               "sample": "a %.0f MiB message of the same recipe (AES-256, 2880-byte AAD): CTR chunked over %d threads, "
                         "GHASH sequential Horner on one" % (sample / 2 ** 20, cores),
               "context": cpu_context(m.key, m.iv)}
        # same leg: the keystream of the sampled blocks of the timed message against the oracle
        from oracle import oracle as O
        for g, got in samples:
            assert np.array_equal(got, np.frombuffer(O.keystream_block(key, m.iv, g), np.uint8)), \
                "keystream block %d differs from the oracle" % g
            verified += 1
    setup["per_call_GBps_including_setup"] = n / ((kernel_ms + setup["gcm_init_wall_ms"]) * 1e-3) / 1e9

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": max(3, args.warmup), "ms_per_step": total_ms / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "u8", "data": "synthetic",
        "config": {"workload": WORKLOAD if n == 4 << 30 else WORKLOAD + " [payload overridden: %d bytes]" % n,
                   "payload_bytes": n, "aad_bytes": int(m.aad.size), "key_bits": 256,
                   "l2": "inputs (4 GiB in + 4 GiB out per step) are larger than the 126 MB L2; no flush needed",
                   "parallelism": "one independent message per GPU, no collective" if world > 1 else "single GPU",
                   "verified_keystream_blocks_vs_oracle": verified},
        "clocks": {k: clocks.get(k) for k in ("sm_mhz", "sm_max_mhz", "reasons", "samples", "power_w_max")},
        "e2e": e2e, "gpu_launches": (3 if uses_tc2 else 1) * args.steps, "roofline": roofline, "cpu_baseline": cpu, "setup": setup,
        "ms_per_step_median": statistics.median(per), "ms_per_step_std": statistics.pstdev(per),
    }
    if world == 1 and not args.no_supplementary and n == 4 << 30:
        del pt, ct
        torch.cuda.empty_cache()
        line["supplementary"] = run_supplementary(args)
    print(json.dumps(line))
    replicas.finish()


# ---------------------------------------------------------------------------------------------------
# supplementary measurements: same timing rules, one JSON line each
# ---------------------------------------------------------------------------------------------------
def run_extra(args):
    import numpy as np
    import torch
    import paper_2602_23067_b200 as G
    import workloads

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(0)
    G.gcm_set_device(0)
    stream = torch.cuda.current_stream()
    peaks = measured_peaks()
    sm_count = torch.cuda.get_device_properties(0).multi_processor_count
    sm_mhz = float(peaks.get("sm_max_mhz", 1965.0))
    w = args.workload
    steps, warm = args.steps, max(3, args.warmup)

    def timed(step):
        for _ in range(warm):
            step()
        torch.cuda.synchronize()
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(steps + 1)]
        sampler = ClockSampler(0)
        sampler.start()
        ev[0].record(stream)
        for i in range(steps):
            step()
            ev[i + 1].record(stream)
        torch.cuda.synchronize()
        clocks = sampler.stop()
        per = [ev[i].elapsed_time(ev[i + 1]) for i in range(steps)]
        return ev[0].elapsed_time(ev[-1]), per, clocks

    def rand_bytes(n, seed):
        gen = torch.Generator(device="cuda")
        gen.manual_seed(seed)
        return torch.randint(-2 ** 63, 2 ** 63 - 1, ((n + 7) // 8,), dtype=torch.int64, device="cuda",
                             generator=gen).view(torch.uint8)[:n]

    line = {"unit": UNIT, "n_gpus": 1, "steps": steps, "warmup": warm, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "u8", "data": "synthetic", "supplementary": True}

    if w in ("c5-decrypt", "c5-ghash", "c5-aes128", "c5-tensor", "c5-aes128-tensor", "c2"):
        n = (256 << 20) if w == "c2" else int(args.size_mib * (1 << 20))
        m = workloads.config_c2(payload_bytes=0) if w == "c2" else workloads.config_c5(payload_bytes=n, with_payload=False)
        key = m.key[:16] if w.startswith("c5-aes128") else m.key
        nr = 10 if len(key) == 16 else 14
        pt = rand_bytes(n, workloads.SEEDS["C2" if w == "c2" else "C5"])
        ct = torch.empty(n, dtype=torch.uint8, device="cuda")
        aad = torch.from_numpy(m.aad).cuda()
        d_tag = torch.zeros(16, dtype=torch.uint8, device="cuda")
        d_status = torch.zeros(1, dtype=torch.int32, device="cuda")
        ctx = G.gcm_init(key)
        if w.endswith("-tensor"):
            G.gcm_set_ghash_engine(ctx, G.GCM_GHASH_TENSOR)     # gcm_tc.cu: the fused kernel with GHASH on the tensor cores
        G.gcm_encrypt_async(ctx, m.iv, aad, pt, ct, d_tag, stream)
        if w == "c5-decrypt":
            back = torch.empty(n, dtype=torch.uint8, device="cuda")
            step = lambda: G.gcm_decrypt_verify_async(ctx, m.iv, aad, ct, back, d_tag, d_status, stream)
            launches, mode, what = 2, "enc", "AES-256-GCM decrypt_verify (fused kernel + gated wipe kernel)"
        elif w == "c5-ghash":
            d_s = torch.zeros(16, dtype=torch.uint8, device="cuda")
            step = lambda: G.gcm_ghash_async(ctx, aad, ct, d_s, stream)
            launches, mode, what = 1, "ghash", "GHASH only over device-resident ciphertext (the paper's Table 5 scope, L363)"
        else:
            step = lambda: G.gcm_encrypt_async(ctx, m.iv, aad, pt, ct, d_tag, stream)
            launches, mode, what = 1, "enc", "AES-%d-GCM encrypt" % (8 * len(key))
        total_ms, per, clocks = timed(step)
        if w == "c5-decrypt":
            assert int(d_status.item()) == 0 and torch.equal(back[:1 << 20], pt[:1 << 20])
        G.gcm_destroy(ctx)
        gbs = steps * n / (total_ms * 1e-3) / 1e9
        key_mix = {"c5-decrypt": "fused_aes256_dec", "c5-ghash": "fused_ghash", "c5-aes128": "fused_aes128_enc", "c2": "fused_aes256_enc",
                   "c5-tensor": "fused_aes256_enc", "c5-aes128-tensor": "fused_aes128_enc"}[w]
        tc2 = mode == "enc" and (w.endswith("-tensor") and n >= (8 << 20) or n >= G.TC2_AUTO_BYTES[128 if nr == 10 else 256])
        if tc2:         # the default engine (or GCM_GHASH_TENSOR) took the gcm_tc2 chain for this size
            key_mix = {"c5-decrypt": "tc2_aes256_dec", "c5-aes128": "tc2_aes128_enc", "c2": "tc2_aes256_enc",
                       "c5-tensor": "tc2_aes256_enc", "c5-aes128-tensor": "tc2_aes128_enc"}[w]
            launches = launches + 2         # the head and tail links of the chain
            what += " (default engine: gcm_tc2 chain, AES warps + tensor-core GHASH)" if not w.endswith("-tensor") else ""
        pb = pipe_bound_gbs(key_mix, nr, sm_count, sm_mhz, G.gcm_measure_pipe_rates(), ghash_only=(mode == "ghash"))
        if w == "c5-ghash":
            # The default engine (GCM_GHASH_AUTO) ran: for a long aligned input that is ONE launch of gcm_ghash_tc_kernel,
            # GHASH as a GF(2) matrix product on tcgen05.mma kind::mxf4 over [pad | AAD | C | length block].  Its bound is the tensor pipe; the table kernel is timed beside it against its own bound.
            ctx = G.gcm_init(key)
            G.gcm_set_ghash_engine(ctx, G.GCM_GHASH_TABLE)
            tab_ms, _, _ = timed(step_with(ctx, aad, ct, stream, G))
            G.gcm_destroy(ctx)
            tab_gbs = steps * n / (tab_ms * 1e-3) / 1e9
            table = roofline_dict(pb, tab_gbs, peaks, 1)
            line.update(metric="%s GB/s (device-timed, %d MiB msg)" % (what, n >> 20), value=gbs, ms_per_step=total_ms / steps,
                        config={"workload": "%s: %s, %d-byte message, 2880-byte AAD; default engine (tensor cores)" % (w, what, n),
                                "payload_bytes": n},
                        gpu_launches=steps, clocks=clocks, roofline=tensor_roofline(gbs, sm_count, sm_mhz, peaks, G.gcm_measure_pipe_rates()),
                        table_engine={"value": tab_gbs, "unit": UNIT, "ms_per_step": tab_ms / steps, "roofline": table},
                        ms_per_step_median=statistics.median(per))
            tpb = line["roofline"].pop("traffic_per_payload_byte", None)
            if tpb is not None:
                line["roofline"]["traffic"] = tpb * n
            return line
        roof = roofline_dict(pb, gbs, peaks, 1 if mode == "ghash" else 2)
        if w.endswith("-tensor") and not tc2:
            # GHASH has left the shared-memory pipe: what binds is the AES table reads alone (the second yardstick);
            # the tcgen05.st / tcgen05.ld traffic of the tensor path adds to it and is not counted here
            y = pb["yardsticks"]
            what += ", GHASH on the tensor cores (gcm_tc.cu)"
            roof.update(peak=y["aes_reads_only_gbs"], frac=gbs / y["aes_reads_only_gbs"],
                        pipe="shared-memory data pipe (LSU): %.1f bank-lanes per block for the AES table reads alone; the multiply "
                             "by K runs on tcgen05.mma kind::mxf4" % y["aes_reads_only_lanes"])
            for k in ("frac_with_global_wavefronts", "counts_per_block", "peak_measured_rates", "frac_measured_rates"):
                roof.pop(k, None)
        line.update(metric="%s GB/s (device-timed, %d MiB msg)" % (what, n >> 20), value=gbs, ms_per_step=total_ms / steps,
                    config={"workload": "%s: %s, %d-byte message, 2880-byte AAD" % (w, what, n), "payload_bytes": n},
                    gpu_launches=launches * steps, clocks=clocks, roofline=roof,
                    ms_per_step_median=statistics.median(per))
    elif w == "c3":
        msgs = workloads.config_c3()
        batch = []
        for m in msgs:
            d_in = torch.from_numpy(m.payload).cuda()
            batch.append({"key": m.key, "iv": m.iv, "aad": torch.from_numpy(m.aad).cuda(), "input": d_in,
                          "output": torch.empty_like(d_in)})
        nbytes = sum(m.payload.size for m in msgs)
        # the gcm_msg array is built once (gcm_pack_msgs), as a C caller's would be; what is timed is the C call
        packed = G.gcm_pack_msgs(batch)
        total_ms, per, clocks = timed(lambda: G.gcm_encrypt_batch(packed, stream))
        G.gcm_batch_release()
        gbs = steps * nbytes / (total_ms * 1e-3) / 1e9
        pb = pipe_bound_gbs("multi_aes256_enc", 14, sm_count, sm_mhz, G.gcm_measure_pipe_rates())
        if not args.no_cpu_baseline:
            line["cpu_baseline"] = oracle_batch_gbs(msgs, "C3")
        line.update(metric="AES-256-GCM batched encrypt GB/s (C3: 16 FITS images of 64 MiB)", value=gbs,
                    ms_per_step=total_ms / steps, gpu_launches=steps, clocks=clocks,
                    config={"workload": "c3: gcm_encrypt_batch, 16 x 67,109,760-byte FITS-shaped images, one AES-256 key, 16 IVs, "
                                        "2880-byte header AAD each; gcm_msg array packed once, synchronous C call (descriptor upload, ONE multi-message launch, tag download inside)",
                            "payload_bytes": nbytes},
                    roofline=roofline_dict(pb, gbs, peaks, 2),
                    ms_per_step_median=statistics.median(per))
    elif w == "c4":
        msgs = workloads.config_c4()
        offs, total = [], 0
        for m in msgs:
            offs.append(total)
            total += (m.payload.size + 15) // 16 * 16
        h_in = np.zeros(total, np.uint8)
        for m, o in zip(msgs, offs):
            h_in[o: o + m.payload.size] = m.payload
        d_in = torch.from_numpy(h_in).cuda()
        d_out = torch.empty_like(d_in)
        aads = [torch.from_numpy(m.aad).cuda() if m.aad.size else None for m in msgs]
        batch = [{"key": m.key, "iv": m.iv, "aad": a, "input": d_in[o: o + m.payload.size],
                  "output": d_out[o: o + m.payload.size]} for m, o, a in zip(msgs, offs, aads)]
        nbytes = sum(m.payload.size for m in msgs)
        # the binding's per-call marshalling of 10,000 Python dicts is host work outside the C ABI:
        # marshal once, then time the C call itself
        packed = G.gcm_pack_msgs(batch)
        arr, cnt, sp = packed.arr, packed.n, G.gcm._stream(stream)

        def step():
            rc = G.gcm._L.gcm_encrypt_batch(arr, cnt, sp)
            assert rc == 0
        total_ms, per, clocks = timed(step)
        # the same batch through the device-descriptor call: descriptors packed and uploaded once, asynchronous launches,
        # nothing marshalled per call (ordering kernel + warp-per-message kernel inside the event pair)
        d_msgs = torch.from_numpy(G.gcm_pack_dmsgs(batch).view(np.uint8).copy()).cuda()
        dev_ms, _, _ = timed(lambda: G.gcm_encrypt_batch_device(d_msgs, len(batch), stream))
        host_tags = bytes(arr[0].tag)
        assert d_msgs.cpu().numpy().view(G.gcm_dmsg_dtype())["tag"][0].tobytes() == host_tags
        line["device_descriptors"] = {"value": steps * nbytes / (dev_ms * 1e-3) / 1e9, "unit": UNIT, "ms_per_step": dev_ms / steps,
                                      "how": "gcm_encrypt_batch_device: gcm_dmsg array resident on the device, asynchronous, device-timed"}
        G.gcm_batch_release()
        gbs = steps * nbytes / (total_ms * 1e-3) / 1e9
        pb = pipe_bound_gbs("batch_aes128_enc", 10, sm_count, sm_mhz, G.gcm_measure_pipe_rates())
        if not args.no_cpu_baseline:
            line["cpu_baseline"] = oracle_batch_gbs(msgs, "C4")
        # C4's latency report: one 1 KiB and one 64 KiB message through the synchronous non-batched call
        lat = {}
        mk = workloads.config_c1(payload_bytes=0)
        lctx = G.gcm_init(mk.key)
        l_aad = torch.from_numpy(mk.aad).cuda()
        for ln in (1024, 65536):
            l_pt = rand_bytes(ln, 7 + ln)
            l_ct = torch.empty_like(l_pt)
            for _ in range(50):
                G.gcm_encrypt(lctx, mk.iv, l_aad, l_pt, l_ct, stream)
            ts = []
            for _ in range(1000):
                t0 = time.perf_counter()
                G.gcm_encrypt(lctx, mk.iv, l_aad, l_pt, l_ct, stream)
                ts.append((time.perf_counter() - t0) * 1e6)
            ts.sort()
            lat["%d_bytes" % ln] = {"p50_us": ts[len(ts) // 2], "p99_us": ts[int(len(ts) * 0.99)]}
        G.gcm_destroy(lctx)
        line["single_message_latency"] = lat
        line.update(metric="AES-128-GCM batched encrypt GB/s (C4: 10,000 messages of 1 B..64 KiB)", value=gbs,
                    ms_per_step=total_ms / steps, gpu_launches=2 * steps, clocks=clocks,
                    messages_per_s=steps * len(msgs) / (total_ms * 1e-3),
                    config={"workload": "c4: gcm_encrypt_batch (C call), 10,000 AES-128 messages, len ~ U{1..65536}, AAD ~ U{0..256}, "
                                        "own key and IV each, payloads packed at 16-byte-aligned offsets; synchronous call "
                                        "(descriptor upload, one persistent warp-per-message kernel, tag download inside)",
                            "payload_bytes": nbytes, "messages": len(msgs)},
                    roofline=dict(roofline_dict(pb, gbs, peaks, 2),
                                  note="the kernel's own mix: 4-bit GHASH table (32 LDS.128 per block) and per-message key "
                                       "schedule, H ladder, table build and tree; achieved is the synchronous C call, host "
                                       "marshalling and transfers included"),
                    ms_per_step_median=statistics.median(per))
    elif w == "datasum":
        # DATASUM reduction kernel (FITS checksum of the encrypted payload): HBM-bound, 1 byte read per byte
        from paper_2602_23067_b200 import gfc
        n = int(args.size_mib * (1 << 20))
        data = rand_bytes(n, 31)
        acc = torch.zeros(1, dtype=torch.int64, device="cuda")
        total_ms, per, clocks = timed(lambda: gfc.gfc_datasum_async(data, acc, stream))
        gbs = steps * n / (total_ms * 1e-3) / 1e9
        hbm = float(peaks["hbm_gbs"])
        line.update(metric="FITS DATASUM kernel GB/s (device-timed, %d MiB)" % (n >> 20), value=gbs, ms_per_step=total_ms / steps,
                    config={"workload": "datasum: 1's-complement sum of big-endian 32-bit words over a %d-byte device buffer "
                                        "(larger than L2; no flush needed)" % n, "payload_bytes": n},
                    gpu_launches=steps, clocks=clocks,
                    roofline={"bound": "hbm", "achieved": gbs, "peak": hbm, "unit": UNIT, "frac": gbs / hbm,
                              "peak_source": "MEASURED_PEAKS.json hbm_gbs (%s)" % peaks["_source"], "traffic": None,
                              "algorithmic_bytes_per_launch": n},
                    ms_per_step_median=statistics.median(per))
    elif w == "frame":
        # The authenticated FITS container end to end (include/gfc.h; PAPER.md sections 3.2.2, 3.3.2, 4.2): host buffers in,
        # host buffers out, header message on streamH concurrently with the chunked data pipeline on streamD.
        from paper_2602_23067_b200 import gfc
        out = {}
        for name, ny, nx in (("256x256", 256, 256), ("4096x4096", 4096, 4096)):
            f = workloads.fits_frame(seed=2100, ny=ny, nx=nx, key_bytes=32, n_sources=50)
            h_fits = torch.frombuffer(bytearray(f.fits), dtype=torch.uint8).pin_memory()
            ctx = gfc.gfc_context_create(16 * 2880, len(f.fits))
            r = gfc.gfc_encrypt_frame(ctx, h_fits, f.key_h, f.key_d, f.nonce_h, f.nonce_d)
            h_cont = torch.from_numpy(r.view().copy()).pin_memory()
            res = {}
            for what, call in (("encrypt", lambda: gfc.gfc_encrypt_frame(ctx, h_fits, f.key_h, f.key_d, f.nonce_h, f.nonce_d)),
                               ("decrypt", lambda: gfc.gfc_decrypt_frame(ctx, h_cont, f.key_h, f.key_d)),
                               ("decrypt_header_only", lambda: gfc.gfc_decrypt_frame(ctx, h_cont, f.key_h, None))):
                for _ in range(warm):
                    call()
                ts, hm, dm = [], [], []
                for _ in range(max(steps, 10)):
                    t0 = time.perf_counter()
                    r = call()
                    ts.append(time.perf_counter() - t0)
                    hm.append(r.header_ms); dm.append(r.data_ms)
                med = statistics.median(ts)
                res[what] = {"wall_ms_median": med * 1e3, "file_GBps": len(f.fits) / med / 1e9,
                             "header_stream_ms": statistics.median(hm), "data_stream_ms": statistics.median(dm),
                             "warning_code": r.warning_code}
            full = gfc.gfc_decrypt_frame(ctx, h_cont, f.key_h, f.key_d)
            assert full.warning_code == 0 and bytes(full.view()[:5760]) == f.fits[:5760]
            gfc.gfc_context_destroy(ctx)
            out[name] = dict(res, file_bytes=len(f.fits))
        big = out["4096x4096"]
        line.update(metric="authenticated FITS container: gfc_decrypt_frame of a 64 MiB image, file GB/s end to end (host wall clock)",
                    value=big["decrypt"]["file_GBps"], ms_per_step=big["decrypt"]["wall_ms_median"],
                    gpu_launches=None, frames=out,
                    config={"workload": "frame: gfc_encrypt_frame / gfc_decrypt_frame (AES-256, dual key) on a 256x256 and a 4096x4096 float32 "
                                        "FITS file in pinned host memory; H2D and D2H inside the timed region (PCIe-bound)"})
    elif w == "sizes":
        # Throughput by message size around the paper's FITS files (17 / 201 / 577 MB, PAPER.md Table A.7): trains of
        # launches back to back on one stream, one event pair around the whole train (an event between two launches
        # costs about 5 us and switches programmatic dependent launch off).
        m = workloads.config_c2(payload_bytes=0)
        ctx = G.gcm_init(m.key)
        aad = torch.from_numpy(m.aad).cuda()
        d_tag = torch.zeros(16, dtype=torch.uint8, device="cuda")
        pb = pipe_bound_gbs("fused_aes256_enc", 14, sm_count, sm_mhz)
        pb2 = pipe_bound_gbs("tc2_aes256_enc", 14, sm_count, sm_mhz)      # from 384 MiB on the default engine runs the gcm_tc2 chain
        out = {}
        for mib in (1, 4, 16, 64, 256, 1024):
            n = mib << 20
            # two buffer pairs used in turn, as a stream of frames would be
            pts = [rand_bytes(n, 200 + mib), rand_bytes(n, 300 + mib)]
            cts = [torch.empty_like(pts[0]), torch.empty_like(pts[1])]
            tags = [torch.zeros(16, dtype=torch.uint8, device="cuda") for _ in range(2)]
            reps = max(steps, 20 if mib >= 256 else 200)
            best = None
            for _ in range(3):
                for i in range(warm):
                    G.gcm_encrypt_async(ctx, m.iv, aad, pts[i & 1], cts[i & 1], tags[i & 1], stream)
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(stream)
                for i in range(reps):
                    G.gcm_encrypt_async(ctx, m.iv, aad, pts[i & 1], cts[i & 1], tags[i & 1], stream)
                e1.record(stream)
                torch.cuda.synchronize()
                us = e0.elapsed_time(e1) * 1e3 / reps
                best = us if best is None else min(best, us)
            tc2 = n >= G.TC2_AUTO_BYTES[256]
            out["%d_MiB" % mib] = {"us_per_launch": best, "GBps": n / best / 1e3, "kernel": "gcm_tc2 chain" if tc2 else "gcm_fused_kernel",
                                   "pipe_bound_gbs": (pb2 if tc2 else pb)["gbs"], "frac_of_pipe_bound": n / best / 1e3 / (pb2 if tc2 else pb)["gbs"]}
            del pts, cts
        G.gcm_destroy(ctx)
        line.update(metric="AES-256-GCM encrypt GB/s by message size (device-timed trains of launches)",
                    value=out["16_MiB"]["GBps"], ms_per_step=out["16_MiB"]["us_per_launch"] / 1e3, gpu_launches=None, sizes=out,
                    roofline={"bound": "alu", "unit_pipe": "lsu_shared", "peak": pb["gbs"], "unit": UNIT,
                              "achieved": out["16_MiB"]["GBps"], "frac": out["16_MiB"]["frac_of_pipe_bound"]},
                    config={"workload": "sizes: AES-256-GCM encrypt of 1 MiB .. 1 GiB device-resident messages, 2880-byte AAD, launches "
                                        "back to back, two buffer pairs in turn; pdl=%s; messages of 16 MiB and less fit in the 126 MB L2 (in + out)"
                                        % ("off" if os.environ.get("GCM_NO_PDL") else "on")})
    elif w == "phases":
        # Where the fixed cost of a launch goes: the fused kernel's own %globaltimer stamps
        # (gcm_set_phase_stamps) for message sizes around the paper's FITS files, launches back to back on one stream.
        m = workloads.config_c2(payload_bytes=0)
        ctx = G.gcm_init(m.key)
        aad = torch.from_numpy(m.aad).cuda()
        d_tag = torch.zeros(16, dtype=torch.uint8, device="cuda")
        grid, _ = G.gcm_get_geometry(ctx)
        stamps = torch.zeros(G.GCM_PHASE_SLOTS * grid, dtype=torch.int64, device="cuda")
        out = {}
        for mib in (1, 4, 16, 64, 256):
            n = mib << 20
            pt = rand_bytes(n, 100 + mib)
            ct = torch.empty_like(pt)
            G.gcm_set_phase_stamps(ctx, None)
            for _ in range(warm):
                G.gcm_encrypt_async(ctx, m.iv, aad, pt, ct, d_tag, stream)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            reps = max(steps, 20)
            e0.record(stream)
            for _ in range(reps):
                G.gcm_encrypt_async(ctx, m.iv, aad, pt, ct, d_tag, stream)
            e1.record(stream)
            torch.cuda.synchronize()
            period_us = e0.elapsed_time(e1) * 1e3 / reps
            # stamps of the LAST of a train of launches (so that its prologue overlaps the previous launch's tail)
            stamps.zero_()
            for _ in range(7):
                G.gcm_encrypt_async(ctx, m.iv, aad, pt, ct, d_tag, stream)
            G.gcm_set_phase_stamps(ctx, stamps)
            G.gcm_encrypt_async(ctx, m.iv, aad, pt, ct, d_tag, stream)
            torch.cuda.synchronize()
            G.gcm_set_phase_stamps(ctx, None)
            st = stamps.cpu().numpy().reshape(grid, G.GCM_PHASE_SLOTS).astype(np.int64)
            live = st[st[:, 0] > 0]
            t0 = live[:, 0].min()
            names = ["entry", "tables_ready", "after_dep_wait", "rows_done", "partials_in", "ticket", "finished", "weights_done"]
            ph = {}
            for k, name in enumerate(names):
                col = live[:, k]
                col = col[col > 0]
                if col.size:
                    ph[name] = {"min_us": float(col.min() - t0) / 1e3, "mean_us": float(col.mean() - t0) / 1e3,
                                "max_us": float(col.max() - t0) / 1e3}
            ph["per_cta_mean_us"] = {
                "entry_to_weights": float((live[:, 7] - live[:, 0]).mean()) / 1e3,
                "entry_to_tables": float((live[:, 1] - live[:, 0]).mean()) / 1e3,
                "tables_to_dep_wait": float((live[:, 2] - live[:, 1]).mean()) / 1e3,
                "rows": float((live[:, 3] - live[:, 2]).mean()) / 1e3,
                "lane_products_and_sync": float((live[:, 4] - live[:, 3]).mean()) / 1e3,
                "cta_combine_and_ticket": float((live[:, 5] - live[:, 4]).mean()) / 1e3,
            }
            out["%d_MiB" % mib] = {"launch_period_us": period_us, "GBps": n / period_us / 1e3, "ctas": int(live.shape[0]),
                                   "first_entry_to_finish_us": ph.get("finished", {}).get("max_us"), "phases": ph}
        G.gcm_destroy(ctx)
        line.update(metric="fused kernel phase breakdown (us, %globaltimer stamps of the last of 8 back-to-back launches)",
                    value=out["16_MiB"]["launch_period_us"], unit="us", higher_is_better=False,
                    ms_per_step=out["16_MiB"]["launch_period_us"] / 1e3, gpu_launches=None, phases=out,
                    config={"workload": "phases: AES-256-GCM encrypt of 1 / 4 / 16 / 64 / 256 MiB, 2880-byte AAD, launches back to back; "
                                        "pdl=%s" % ("off" if os.environ.get("GCM_NO_PDL") else "on")})
    elif w == "latency":
        # single-message latency through the synchronous non-batched call (C4's report): host wall clock
        m = workloads.config_c1(payload_bytes=0)
        ctx = G.gcm_init(m.key)
        aad = torch.from_numpy(m.aad).cuda()
        out = {}
        for n in (1024, 65536, 1 << 20):
            pt = rand_bytes(n, 7 + n)
            ct = torch.empty_like(pt)
            for _ in range(50):
                G.gcm_encrypt(ctx, m.iv, aad, pt, ct, stream)
            ts = []
            for _ in range(2000):
                t0 = time.perf_counter()
                G.gcm_encrypt(ctx, m.iv, aad, pt, ct, stream)
                ts.append((time.perf_counter() - t0) * 1e6)
            ts.sort()
            out["%d_bytes" % n] = {"p50_us": ts[len(ts) // 2], "p99_us": ts[int(len(ts) * 0.99)], "min_us": ts[0]}
        G.gcm_destroy(ctx)
        line.update(metric="AES-128-GCM single-message latency through gcm_encrypt (us, host wall clock)", value=out["1024_bytes"]["p50_us"],
                    unit="us", higher_is_better=False, ms_per_step=out["1024_bytes"]["p50_us"] / 1e3, gpu_launches=2000 * 3,
                    config={"workload": "latency: synchronous gcm_encrypt of one 1 KiB / 64 KiB / 1 MiB AES-128 message, 16-byte AAD, 2000 calls each"},
                    latency=out)
    return line


# The supplementary workloads that ride in the default line (BASELINE.json configs 2-4, the decrypt direction, AES-128,
# GHASH only as in PAPER.md Table 5, the by-size sweep around the paper's file sizes of Table A.7, call latency), with
# the timed steps each gets there.  Same code as `--workload <name>`, which prints the full line of each.
SUPPLEMENTARY = [("c2", 20), ("c3", 10), ("c4", 20), ("c5-decrypt", 10), ("c5-aes128", 10), ("c5-ghash", 10), ("sizes", 20), ("latency", 1)]


def run_supplementary(args) -> dict:
    """{workload: compact result} for the default line's `supplementary` object; a workload that fails is recorded as
    {"error": ...} and does not take the headline down with it."""
    import argparse
    out = {}
    t_all = time.perf_counter()
    for w, k in SUPPLEMENTARY:
        sub = argparse.Namespace(**{**vars(args), "workload": w, "steps": k, "warmup": 3, "no_cpu_baseline": True})
        t0 = time.perf_counter()
        try:
            ln = run_extra(sub)
        except BaseException as e:                     # SystemExit of a missing mix entry included
            out[w] = {"error": "%s: %s" % (type(e).__name__, e)}
            continue
        r = ln.get("roofline") or {}
        c = {"metric": ln.get("metric"), "value": ln.get("value"), "unit": ln.get("unit"), "steps": ln.get("steps"),
             "ms_per_step": ln.get("ms_per_step"), "gpu_launches": ln.get("gpu_launches"),
             "roofline": {k2: r.get(k2) for k2 in ("bound", "unit_pipe", "peak", "frac", "unit", "frac_of_aes_reads_only_floor",
                                                    "frac_of_mma_issue_rate", "kernel") if r.get(k2) is not None},
             "sm_mhz": (ln.get("clocks") or {}).get("sm_mhz"), "wall_s": round(time.perf_counter() - t0, 1)}
        for extra in ("device_descriptors", "single_message_latency", "latency", "sizes", "messages_per_s"):
            if extra in ln:
                c[extra] = ln[extra]
        if isinstance(ln.get("table_engine"), dict):
            c["table_engine"] = {k2: ln["table_engine"].get(k2) for k2 in ("value", "unit", "ms_per_step")}
        out[w] = c
    out["wall_s"] = round(time.perf_counter() - t_all, 1)
    return out


def main():
    args = parse_args()
    if args.impl == "reference":
        run_reference(args)
    elif args.workload == "c5":
        run_ours(args)
    else:
        print(json.dumps(run_extra(args)))


if __name__ == "__main__":
    main()
