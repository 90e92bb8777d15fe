"""bench.py -- lineal path function throughput on B200 (segment tests/s) and ALU roofline fraction.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg3|cfg4|cfg2] [--flags prune,notrie]
    python bench.py --impl reference ...      # the CPU oracle as it stands, bounded sample per step

A step is one pass of the whole hot path (bit-pack + stage, trie walk, count, mirror,
and for cfg4 the objective) over one batch of synthetic images already resident in HBM.  Nominal
segment tests of a step = B * n_phases * H * W * (2m+1)^2.  The L2 is flushed
(256 MiB memset) between timed steps, outside the per-step CUDA-event pairs; the reported time is
the sum of the K per-step device times, max over ranks.  N > 1: one process per GPU, each rank
evaluates its own independent images (weak scaling, no data-path collective)."""
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
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_1601_04359_b200 import inputs  # noqa: E402  (seeded generators only; no method arithmetic)
from paper_1601_04359_b200 import dist as lpf_dist  # noqa: E402  (rank plumbing: seeds, max over ranks)

METRIC = "segment tests/sec (start-pixel x vector)"
UNIT = "segment tests/s"
SM_COUNT = 148
ALU_LANES_PER_CLK_PER_SM = 64     # 4 sub-partitions x 16 lanes: alu pipe issues one warp instruction per 2 clk
                                  # per sub-partition (B300_MICROARCH.md "Pipe rates": rt_SMSP = 2)

WORKLOADS = {
    # name: (config number, H, W, m, phases, images per rank)
    "cfg2": dict(cfg=2, H=256, W=256, m=128, n_phase=2, B=1),
    "cfg3": dict(cfg=3, H=512, W=512, m=256, n_phase=2, B=1),
    "cfg4": dict(cfg=4, H=128, W=128, m=64, n_phase=1, B=1024),
}


def make_images(w, rank):
    """Synthetic images of the workload for this rank (rank r offsets the seed by 100000 r)."""
    c = w["cfg"]
    off = lpf_dist.rank_seed_offset(rank)
    if c == 2:
        return inputs.disks(256, 256, 8.0, 0.30, inputs.seed_for(2) + off)[None], None
    if c == 3:
        return inputs.gaussian_field(512, 512, 12.0, 0.40, inputs.seed_for(3) + off)[None], None
    B = w["B"]
    imgs = np.stack([inputs.disks(128, 128, 6.0, 0.35, inputs.seed_for(4, i) + off) for i in range(B)])
    target = inputs.disks(128, 128, 6.0, 0.35, inputs.seed_for(4, B) + off)
    return imgs, target


def nominal_tests(w):
    S = 2 * w["m"] + 1
    return w["B"] * w["n_phase"] * w["H"] * w["W"] * S * S


def survey_ops(w, info):
    """SURVEY.md 8(d)'s op model: per image-phase Nw * (2 * trie nodes + 2 * half vectors) -- (SHF + LOP3) per word-node,
    (POPC + add) per word-terminal.  The design needs fewer (below), so this is kept as a secondary figure only."""
    nw = w["H"] * w["W"] // 32
    return w["B"] * w["n_phase"] * nw * (2 * info["n_trie_nodes"] + 2 * info["n_half_vectors"])


def design_ops(w, launch):
    """Data operations the DESIGN executes at minimum, from the program that was actually uploaded (replayed on the host
    by the library, lpf_last_launch_info): per image-phase and per start word, a fused pair of entries costs 2 SHF + 1
    LOP3, an entry on its own 1 SHF + 1 LOP3, a terminal 1 POPC + 1 add.  Times the H*W/32 start words of an image
    (not the padded strips), images and phases.  Overhead instructions (loads, entry decode, reductions) are not counted:
    this is the numerator of a utilisation, so it is <= the ALU pipe's executed count."""
    nw = w["H"] * w["W"] // 32
    per_word = 3 * launch["fused_pairs"] + 2 * launch["singles"] + 2 * launch["terminals"]
    return w["B"] * w["n_phase"] * nw * per_word


def design_smem_bytes(w, launch):
    """Shared-memory bytes the DESIGN loads at minimum: an entry that changes row, word column or plane reloads its row
    strip, TY * (TX + 1) words per thread for TX * TY start words (tile code = 1000 TX + 100 TY + slots), i.e.
    (TX + 1) / TX words per start word; counted from the uploaded program (`reloads`), times start words, images, phases."""
    tx = launch["tile"] // 1000
    nw = w["H"] * w["W"] // 32
    return w["B"] * w["n_phase"] * nw * launch["reloads"] * (tx + 1) / tx * 4.0


def csrc_digest():
    """sha256 over the CUDA/C++ sources and the public header: the key of profiles/capture_index.csv, so that ncu
    figures are only quoted for the kernels they were captured from."""
    import hashlib
    h = hashlib.sha256()
    csrc = os.path.join(ROOT, "paper_1601_04359_b200", "csrc")
    for name in sorted(os.listdir(csrc)) + [os.path.join("..", "..", "include", "lpf.h")]:
        with open(os.path.join(csrc, name), "rb") as f:
            h.update(name.encode() + b"\0" + f.read())
    return h.hexdigest()[:16]


def capture_lookup(workload, flags):
    """ncu figures of the eval kernel for (these sources, workload, flags) from profiles/capture_index.csv, or None."""
    import csv
    path = os.path.join(ROOT, "profiles", "capture_index.csv")
    if not os.path.exists(path):
        return None
    key = csrc_digest()
    for row in csv.DictReader(open(path)):
        if row["csrc_sha256"] == key and row["workload"] == workload and row["flags"] == (flags or "none"):
            out = {k: float(row[k]) for k in ("alu_pipe_pct", "smem_wavefront_pct", "issue_active_pct",
                                              "dram_read_bytes", "dram_write_bytes", "gpu_time_us")}
            out["source"] = row["source"]
            return out
    return None


class ClockSampler(threading.Thread):
    """nvidia-smi clocks/throttle reasons sampled during the timed region (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index = index
        self.rows = []
        self.proc = None

    def run(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            for line in self.proc.stdout:
                self.rows.append([t.strip() for t in line.split(",")])
        except Exception:
            pass

    def stop(self):
        if self.proc is not None:
            self.proc.terminate()
        self.join(timeout=2)
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0]))
                mx.append(float(r[1]))
                for n, v in zip(names, r[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(n)
            except Exception:
                continue
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def oracle_sample(w, imgs, seconds_hint, rng_seed=0, n_vec=None, threads=None):
    """The oracle as it stands on a bounded sample of the workload: a random subset of template vectors
    (all start pixels, all phases of the workload) on the first image. Returns (tests, seconds, cores, what)."""
    from oracle import lpf_oracle as orc
    m = w["m"]
    rng = np.random.default_rng(rng_seed)
    if n_vec is None:
        n_vec = {2: 24000, 3: 6000, 4: 80000}[w["cfg"]]      # about 15 s on 16 cores
    vecs = rng.integers(-m, m + 1, size=(n_vec, 2))
    img = imgs[0]
    t0 = time.perf_counter()
    cores = 1
    for phase in ((0, 1) if w["n_phase"] == 2 else (1,)):
        # all host cores by default, whatever OMP_NUM_THREADS torchrun set
        _, cores = orc.counts_list(img, phase, vecs, threads=threads or os.cpu_count() or 1)
    dt = time.perf_counter() - t0
    tests = n_vec * w["H"] * w["W"] * w["n_phase"]
    what = "%d random template vectors x all %dx%d start pixels x %d phase(s) of image 0" % (
        n_vec, w["H"], w["W"], w["n_phase"])
    return tests, dt, cores, what


def run_reference(args, w, rank, world):
    """--impl reference: the CPU oracle (oracle/), unmodified, on the host cores; rank 0 only."""
    if rank != 0:
        return
    imgs, _ = make_images(w, 0)
    total_tests, total_s, cores, what = 0, 0.0, 1, ""
    for i in range(args.warmup + args.steps):
        tests, dt, cores, what = oracle_sample(w, imgs, 0, rng_seed=i, n_vec={2: 2000, 3: 400, 4: 6000}[w["cfg"]])
        if i >= args.warmup:
            total_tests += tests
            total_s += dt
    value = total_tests / total_s
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * total_s / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "u8", "data": "synthetic",
            "config": {"workload": args.workload_desc, "sample_per_step": what},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": what},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


TAB1_SIZES = (10, 20, 50, 100, 200, 500)
# paper's Tab. 1, standard / enhanced GPU seconds on a Quadro 4000, both phases; context only
TAB1_PAPER = {"chess": {10: (2.4e-3, 2.4e-3), 20: (11.9e-3, 11.1e-3), 50: (0.15, 0.10), 100: (2.1, 0.26),
                        200: (32.6, 2.0), 500: (318.4, 16.3)},
              "squares": {10: (2.5e-3, 2.5e-3), 20: (12.9e-3, 12.5e-3), 50: (0.16, 0.13), 100: (2.5, 1.7),
                          200: (41.9, 20.8), 500: (411.6, 205.1)}}


def run_tab1(lpf, torch, device, out_dir):
    """Tab. 1-shaped study: one evaluation of the ENTIRE L2 (all segments up to
    W-1, H-1, i.e. m = size - 1) for both phases, standard and enhanced (LPF_PRUNE), on the two morphologies the
    paper describes in words: chess with 10x10 px fields and a suspension of 4x4 px squares (its volume fraction is
    not printed; 0.20 here).  Times: eval kernel alone, whole device step, and the paper's quantity -- host image in,
    host counts out (Alg. 2 lines 6-21) -- through lpf_eval_host, mean of 5 after one warm-up.  Every cell is checked
    bit-exactly against the CPU oracle on 200 random vectors per phase.  Returns a list of row dicts."""
    from oracle import lpf_oracle as orc
    rows = []
    for size in TAB1_SIZES:
        m = size - 1
        p = lpf.lpf_build_paths(m, device)                    # paper step 1: untimed
        lpf.lpf_set_timing(p, True)
        for morph in ("chess", "squares"):
            img = inputs.chess(size, size, 10) if morph == "chess" else \
                inputs.squares(size, size, 4, 0.20, inputs.seed_for(6, size))
            d_img = torch.from_numpy(img[None]).cuda()
            h_in = torch.from_numpy(img[None].copy()).pin_memory()
            S = 2 * m + 1
            h_out = torch.empty((1, 2, S, S), dtype=torch.int64).pin_memory()
            rng = np.random.default_rng(size)
            vecs = rng.integers(-m, m + 1, size=(200, 2))
            row = {"morphology": morph, "size": size, "segments": 2 * m * m + 2 * m + 1,
                   "paper_gpu_s": TAB1_PAPER[morph][size]}
            for name, flags in (("standard", 0), ("enhanced", lpf.LPF_PRUNE)):
                out = lpf.lpf_eval_both(p, d_img, flags)
                torch.cuda.synchronize()
                c = out.cpu().numpy()[0]
                for phase in (0, 1):
                    want, _ = orc.counts_list(img, phase, vecs)
                    got = c[phase][vecs[:, 1] + m, vecs[:, 0] + m]
                    if not np.array_equal(got, want):
                        raise AssertionError("tab1: %s %d %s phase %d differs from the oracle" % (morph, size, name, phase))
                ker, dev_ms = [], []
                for _ in range(5):
                    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    e0.record()
                    lpf.lpf_eval_both(p, d_img, flags, out=out)
                    e1.record()
                    torch.cuda.synchronize()
                    dev_ms.append(e0.elapsed_time(e1))
                    ker.append(lpf.lpf_last_eval_kernel_ms(p))
                lpf.lpf_eval_host(p, h_in, -1, h_out, flags)
                t0 = time.perf_counter()
                for _ in range(5):
                    lpf.lpf_eval_host(p, h_in, -1, h_out, flags)
                e2e = (time.perf_counter() - t0) / 5
                row[name] = {"kernel_ms": float(np.mean(ker)), "device_ms": float(np.mean(dev_ms)), "e2e_s": e2e}
            rows.append(row)
            print("tab1 %-8s %4d  std %.3f ms  enh %.3f ms  e2e %.3f / %.3f ms" % (
                morph, size, row["standard"]["device_ms"], row["enhanced"]["device_ms"],
                1e3 * row["standard"]["e2e_s"], 1e3 * row["enhanced"]["e2e_s"]), file=sys.stderr, flush=True)
        lpf.lpf_free_paths(p)
    os.makedirs(out_dir, exist_ok=True)
    with open(os.path.join(out_dir, "tab1.json"), "w") as f:
        json.dump(rows, f, indent=1)
    with open(os.path.join(out_dir, "tab1.md"), "w") as f:
        f.write("| morphology | size | segments | std kernel ms | std e2e ms | enh kernel ms | enh e2e ms | "
                "paper GPU std s | paper GPU enh s | e2e speed-up std | enh |\n|---|---|---|---|---|---|---|---|---|---|---|\n")
        for r in rows:
            ps, pe = r["paper_gpu_s"]
            f.write("| %s | %d | %d | %.3f | %.3f | %.3f | %.3f | %g | %g | %.0fx | %.0fx |\n" % (
                r["morphology"], r["size"], r["segments"], r["standard"]["kernel_ms"], 1e3 * r["standard"]["e2e_s"],
                r["enhanced"]["kernel_ms"], 1e3 * r["enhanced"]["e2e_s"], ps, pe,
                ps / r["standard"]["e2e_s"], pe / r["enhanced"]["e2e_s"]))
    return rows


FIG7_N = (100, 200, 500, 1000, 2000, 4000, 6000, 8000, 9000, 9500, 10000)


def run_fig7(lpf, torch, device, out_dir):
    """Fig. 7-shaped study: error of the N-position approximation L2~ of the
    lineal path function against the exact L2, Eq. 14: e = sum over D of (L2 - L2~)^2, as a function of the number N of
    start positions, drawn as a random N-combination WITHOUT repetition, on three 100 x 100 images (the paper's three
    are not in the container: a chess board with 10 px fields, a suspension of 4 x 4 squares and a disk model stand in),
    entire domain (m = 99), both phases.  L2 = counts / (W H), L2~ = masked counts / N.  e must be exactly 0 at
    N = W H.  One point per image is re-checked against the CPU oracle in the run."""
    from oracle import lpf_oracle as orc
    H = W = 100
    m = 99
    S = 2 * m + 1
    p = lpf.lpf_build_paths(m, device)
    lpf.lpf_reserve(p, 1, H, W, 0, lpf.LPF_FOR_EVAL_BOTH)
    lpf.lpf_reserve(p, 1, H, W, 0, lpf.LPF_FOR_EVAL_BOTH | lpf.LPF_FOR_MASKED)
    half = (torch.arange(S * S, device="cuda") >= m * S + m).reshape(S, S)        # D of Eq. 13
    images = {"chess 10 px": inputs.chess(H, W, 10), "squares 4 px, 0.20": inputs.squares(H, W, 4, 0.20, inputs.seed_for(6, 100)),
              "disks r = 8, 0.45": inputs.disks(H, W, 8.0, 0.45, inputs.seed_for(10))}
    rows = []
    for name, img in images.items():
        d_img = torch.from_numpy(img[None]).cuda()
        exact = lpf.lpf_eval_both(p, d_img)[0].double() / (W * H)
        rng = np.random.default_rng(inputs.seed_for(10, 1))
        order = rng.permutation(H * W)                        # nested N-combinations without repetition
        for N in FIG7_N:
            mask = np.zeros(H * W, dtype=np.uint8)
            mask[order[:N]] = 1
            d_mask = torch.from_numpy(mask.reshape(H, W)).cuda()
            got = lpf.lpf_eval_masked(p, d_img, -1, d_mask)[0]
            err = (((exact - got.double() / N) ** 2) * half).sum(dim=(1, 2)).cpu().numpy()
            rows.append({"image": name, "N": N, "e_phase0": float(err[0]), "e_phase1": float(err[1])})
            if N == 1000:                                     # spot check of the masked counts against the oracle
                vecs = rng.integers(-m, m + 1, size=(60, 2))
                vecs = np.array([v if (v[1] > 0 or (v[1] == 0 and v[0] >= 0)) else -v for v in vecs])
                for ph in (0, 1):
                    want = orc.counts_masked(img, mask.reshape(H, W), ph, vecs)
                    if not np.array_equal(got[ph].cpu().numpy()[vecs[:, 1] + m, vecs[:, 0] + m], want):
                        raise AssertionError("fig7: masked counts differ from the oracle (%s, phase %d)" % (name, ph))
        if rows[-1]["e_phase0"] != 0.0 or rows[-1]["e_phase1"] != 0.0:
            raise AssertionError("fig7: the error at N = WH is not zero")
    lpf.lpf_free_paths(p)
    os.makedirs(out_dir, exist_ok=True)
    with open(os.path.join(out_dir, "fig7.json"), "w") as f:
        json.dump(rows, f, indent=1)
    with open(os.path.join(out_dir, "fig7.md"), "w") as f:
        f.write("| image (100 x 100, m = 99) | N | e(L2, phase 0) | e(L2, phase 1) |\n|---|---|---|---|\n")
        for r in rows:
            f.write("| %s | %d | %.4e | %.4e |\n" % (r["image"], r["N"], r["e_phase0"], r["e_phase1"]))
    return rows


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg3", choices=sorted(WORKLOADS))
    ap.add_argument("--flags", default="")
    ap.add_argument("--scaling", default="weak", choices=["weak", "strong"],
                    help="N > 1: weak = every rank evaluates its own full workload; strong (cfg4) = the ONE batch of 1024 "
                         "images is split over the ranks (PAPER.md:353) and the count slices are all-gathered")
    ap.add_argument("--fig7", action="store_true",
                    help="also run the Fig. 7-shaped study of the N-position approximation (PAPER.md:160-172) and write "
                         "gpurun_out/fig7.{json,md}")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-extra", action="store_true", help="skip the secondary workloads in the same JSON line")
    ap.add_argument("--leg", default="", choices=["", "cfg5", "anneal", "s2", "ensemble"],
                    help="run ONE secondary leg alone and print its JSON (used for the ncu captures under profiles/)")
    ap.add_argument("--tab1", action="store_true",
                    help="also run the Tab. 1-shaped size study (chess / 4x4 squares, 10..500 px, m = size - 1) and "
                         "write gpurun_out/tab1.{json,md}")
    args = ap.parse_args()
    w = WORKLOADS[args.workload]
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    S = 2 * w["m"] + 1
    args.workload_desc = "config %d: %d x %dx%d periodic image(s), %d phase(s), template |dx|,|dy|<=%d (%d vectors)" % (
        w["cfg"], w["B"], w["H"], w["W"], w["n_phase"], w["m"], S * S)
    if args.impl == "reference":
        run_reference(args, w, rank, world)
        return

    import torch
    import torch.distributed as dist
    from paper_1601_04359_b200 import build as lpf_build
    from paper_1601_04359_b200 import lpf

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback")
    lpf_build.build()
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    flags = 0
    for f in [t for t in args.flags.split(",") if t]:
        flags |= {"prune": lpf.LPF_PRUNE, "notrie": lpf.LPF_NO_TRIE}[f]

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    def measure(wl, steps, warmup, with_e2e, strong=False, level=-1):
        """Times `steps` steps of workload wl. Returns dict of results for this rank (max over ranks applied).
        strong: all ranks hold the same batch, rank r evaluates the images lpf_dist.shard_range(B, r, world) and the
        per-rank count slices are all-gathered (the one collective of the split path) inside the timed region."""
        strong = strong and world > 1 and wl["B"] >= world
        imgs, target_img = make_images(wl, 0 if strong else rank)
        b0, b1 = lpf_dist.shard_range(wl["B"], rank, world) if strong else (0, wl["B"])
        imgs = imgs[b0:b1]
        B_loc = b1 - b0
        p = lpf.lpf_build_paths(wl["m"], local_rank)      # paper step 1: untimed
        lpf.lpf_set_level(p, level)                       # -1: automatic (the design variants cap the erosion level)
        info = lpf.lpf_paths_info(p)
        d_imgs = torch.from_numpy(imgs).cuda()
        Sw = 2 * wl["m"] + 1
        shape = (B_loc, 2, Sw, Sw) if wl["n_phase"] == 2 else (B_loc, Sw, Sw)
        d_counts = torch.empty(shape, dtype=torch.int64, device="cuda")
        d_all = lpf_dist.gather_buffer(d_counts, wl["B"], world) if strong else None
        d_target = d_sse = None
        if target_img is not None:
            d_target = lpf.lpf_eval(p, torch.from_numpy(target_img[None]).cuda(), 1)[0].clone()
            d_sse = torch.empty((B_loc,), dtype=torch.int64, device="cuda")
        flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
        stream = torch.cuda.current_stream()
        lpf.lpf_reserve(p, B_loc, wl["H"], wl["W"], flags,
                        (lpf.LPF_FOR_EVAL_BOTH if wl["n_phase"] == 2 else lpf.LPF_FOR_EVAL) | lpf.LPF_FOR_HOST)
        lpf.lpf_set_timing(p, True)

        def step():
            if wl["n_phase"] == 2:
                lpf.lpf_eval_both(p, d_imgs, flags, out=d_counts, stream=stream)
            else:
                lpf.lpf_eval(p, d_imgs, 1, flags, out=d_counts, stream=stream)
            if d_target is not None:
                lpf.lpf_objective(d_counts, d_target, out=d_sse, stream=stream)
            if strong:                                    # every rank ends the step with the whole [B, S, S] array
                lpf_dist.gather_shards(d_counts, d_all, wl["B"], rank, world)

        for _ in range(warmup):
            flush.zero_()
            step()
        barrier()
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        kernel_ms = []
        sampler = ClockSampler(local_rank) if (rank == 0 and with_e2e) else None
        if sampler:
            sampler.start()
            time.sleep(0.3)
        wall0 = time.perf_counter()
        for i in range(steps):
            flush.zero_()                         # L2 flush between timed iterations, outside the event pair
            ev[i][0].record(stream)
            step()
            ev[i][1].record(stream)
            kernel_ms.append(None)
            ev[i][1].synchronize()
            kernel_ms[i] = lpf.lpf_last_eval_kernel_ms(p)
        barrier()
        wall = time.perf_counter() - wall0
        clocks = sampler.stop() if sampler else None
        step_ms = [a.elapsed_time(b) for a, b in ev]
        total_ms = float(sum(step_ms))
        launch = lpf.lpf_last_launch_info(p)
        launches_per_step = launch["kernels"] + (1 if d_target is not None else 0)

        # end to end through the C ABI with HOST buffers: pinned input -> H2D -> hot path -> D2H of the counts
        e2e = None
        if with_e2e:
            h_in = torch.from_numpy(imgs).pin_memory()
            h_out = torch.empty(shape, dtype=torch.int64).pin_memory()
            phase_arg = -1 if wl["n_phase"] == 2 else 1
            k = max(3, min(steps, 5))
            lpf.lpf_eval_host(p, h_in, phase_arg, h_out, flags)
            barrier()
            t0 = time.perf_counter()
            for _ in range(k):
                lpf.lpf_eval_host(p, h_in, phase_arg, h_out, flags)
            torch.cuda.synchronize()
            e2e_s = (time.perf_counter() - t0) / k
            e2e = {"seconds_per_step": e2e_s, "h2d": int(h_in.numel()), "d2h": int(h_out.numel() * 8)}
        total_ms, kern_ms, e2e_s = lpf_dist.max_over_ranks(
            [total_ms, float(np.mean(kernel_ms)), e2e["seconds_per_step"] if e2e else 0.0], device="cuda")
        lpf.lpf_free_paths(p)
        return dict(total_ms=total_ms, kernel_ms=kern_ms, e2e_s=e2e_s, e2e=e2e, info=info, launch=launch,
                    launches_per_step=launches_per_step, clocks=clocks, imgs=imgs, wall=wall, images_per_gpu=B_loc,
                    strong=strong)

    def measure_swaps(n=20000):
        """config 5: n independent two-pixel swap proposals on the 256x256 disk image, m = 64; phase 1 (the config) and,
        on a quarter of the proposals, phase 0 (the matrix: long in-phase segments, a much larger live region)."""
        img = inputs.config_image(5)
        pairs = inputs.config5_pairs(img, 2 * n)
        p5 = lpf.lpf_build_paths(64, local_rank)
        info5 = lpf.lpf_paths_info(p5)
        lpf.lpf_reserve(p5, 1, 256, 256, 0, lpf.LPF_FOR_SWAP_DELTA)
        d_img = torch.from_numpy(img[None]).cuda()
        d_pairs = torch.from_numpy(pairs).cuda()
        out = torch.empty((n, 129, 129), dtype=torch.int32, device="cuda")
        cand = 2 * (2 * info5["sum_path_len"] - 1)          # candidate (start, vector) tests per swap, SURVEY 8 a9
        res = {}
        for phase, k in ((1, n), (0, n // 4)):
            lpf.lpf_swap_delta(p5, d_img, phase, d_pairs[:k], out=out[:k])
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            lpf.lpf_swap_delta(p5, d_img, phase, d_pairs[n:n + k], out=out[:k])
            e1.record()
            torch.cuda.synchronize()
            ms = e0.elapsed_time(e1)
            res["phase%d" % phase] = {"swaps": k, "ms": ms, "swaps_per_s": k / (ms * 1e-3),
                                      "candidate_tests_per_s": k * cand / (ms * 1e-3),
                                      "d2d_bytes_out": int(k * 129 * 129 * 4)}
        lpf.lpf_free_paths(p5)
        res.update(res["phase1"])                            # the config's own figures at the top level
        return res

    def measure_s2(cfg_name):
        """Two-point probability of both phases (LPF_S2: exact integer counts of Eq. 6, O(WH * S^2) bit operations) on a
        workload's image, next to the transform form of Eq. 7 (O(WH log WH), floating point) run with
        torch.fft = cuFFT on the same image as CONTEXT -- it is a library call and not part of this library's path."""
        wl = WORKLOADS[cfg_name]
        imgs, _ = make_images(wl, 0)
        p2 = lpf.lpf_build_paths(wl["m"], local_rank)
        lpf.lpf_reserve(p2, 1, wl["H"], wl["W"], lpf.LPF_S2, lpf.LPF_FOR_EVAL_BOTH)
        lpf.lpf_set_timing(p2, True)
        d_img = torch.from_numpy(imgs[:1]).cuda()
        out = lpf.lpf_eval_both(p2, d_img, lpf.LPF_S2)
        torch.cuda.synchronize()
        step_ms, ker_ms = [], []
        for _ in range(5):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            lpf.lpf_eval_both(p2, d_img, lpf.LPF_S2, out=out)
            e1.record()
            torch.cuda.synchronize()
            step_ms.append(e0.elapsed_time(e1))
            ker_ms.append(lpf.lpf_last_eval_kernel_ms(p2))
        m = wl["m"]

        def fft_form():
            chi = torch.stack([(d_img[0] == 0), (d_img[0] == 1)]).to(torch.float64)
            F = torch.fft.rfft2(chi)
            return torch.fft.irfft2(F * F.conj(), s=chi.shape[-2:])
        corr = fft_form()
        torch.cuda.synchronize()
        fft_ms = []
        for _ in range(5):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            corr = fft_form()
            e1.record()
            torch.cuda.synchronize()
            fft_ms.append(e0.elapsed_time(e1))
        idx = (-torch.arange(-m, m + 1, device="cuda")) % wl["H"]
        jdx = (-torch.arange(-m, m + 1, device="cuda")) % wl["W"]
        same = bool((torch.round(corr[:, idx][:, :, jdx]).to(torch.int64) == out[0]).all())
        lpf.lpf_free_paths(p2)
        return {"direct_step_ms": float(np.median(step_ms)), "direct_kernel_ms": float(np.median(ker_ms)),
                "cufft_context_ms": float(np.median(fft_ms)), "direct_over_cufft": float(np.median(step_ms) / np.median(fft_ms)),
                "rounded_fft_equals_exact_counts": same}

    def measure_ensemble():
        """lpf_eval_sum: ensemble descriptor of 100 slices of 100 x 100, both phases, entire L2
        (m = 99), against the per-image call + a device-side sum over the batch."""
        B, H, W, m = 100, 100, 100, 99
        stack = np.stack([inputs.disks(H, W, 5.0, 0.45, inputs.seed_for(9, i)) for i in range(B)])
        pe = lpf.lpf_build_paths(m, local_rank)
        lpf.lpf_reserve(pe, B, H, W, 0, lpf.LPF_FOR_EVAL_BOTH)
        d = torch.from_numpy(stack).cuda()
        out = lpf.lpf_eval_sum(pe, d, -1)
        per = lpf.lpf_eval_both(pe, d)
        ok = bool((per.sum(dim=0) == out).all())
        torch.cuda.synchronize()
        t_sum, t_per = [], []
        for _ in range(5):
            e0, e1, e2 = (torch.cuda.Event(enable_timing=True) for _ in range(3))
            e0.record()
            lpf.lpf_eval_sum(pe, d, -1, out=out)
            e1.record()
            lpf.lpf_eval_both(pe, d, out=per)
            per.sum(dim=0)
            e2.record()
            torch.cuda.synchronize()
            t_sum.append(e0.elapsed_time(e1))
            t_per.append(e1.elapsed_time(e2))
        lpf.lpf_free_paths(pe)
        S = 2 * m + 1
        return {"slices": B, "eval_sum_ms": float(np.median(t_sum)), "per_image_then_sum_ms": float(np.median(t_per)),
                "equal": ok, "tests_per_s": B * 2 * H * W * S * S / (np.median(t_sum) * 1e-3)}

    def measure_anneal(n=20000):
        """Alg. 3 (lpf_anneal) on the paper's compression setting: target = descriptor of a 100x100
        suspension of 4x4 squares, start = its pixels shuffled, both phases, m = 49, Tab. 2 ratios for c_max, s_max."""
        H = W = 100
        m = 49
        tgt_img = inputs.squares(H, W, 4, 0.20, inputs.seed_for(7))
        start = tgt_img.flatten()
        np.random.default_rng(inputs.seed_for(7, 1)).shuffle(start)
        pairs, log_u = inputs.anneal_proposals(H, W, n, inputs.seed_for(7, 2))
        pa = lpf.lpf_build_paths(m, local_rank)
        lpf.lpf_reserve(pa, 1, H, W, 0, lpf.LPF_FOR_ANNEAL)
        target = lpf.lpf_eval_both(pa, torch.from_numpy(tgt_img[None]).cuda())[0].clone()
        d_img = torch.from_numpy(start.reshape(1, H, W).copy()).cuda()
        c0 = lpf.lpf_eval_both(pa, d_img)[0]
        half = torch.arange((2 * m + 1) ** 2, device="cuda").reshape(2 * m + 1, 2 * m + 1) >= (m * (2 * m + 1) + m)
        E0 = float((((target - c0)[:, half]) ** 2).sum())
        # T_max so that a typical worsening move is accepted with probability 1/2 at the start (Tab. 2: "s/c = 0.5"):
        # pilot of 256 proposals against the start image
        d_pairs = torch.from_numpy(pairs).cuda()
        dE = torch.zeros(256, dtype=torch.int64, device="cuda")
        for ph in (0, 1):
            dl = lpf.lpf_swap_delta(pa, d_img, ph, d_pairs[:256]).to(torch.int64)[:, half]
            dd = (target[ph] - c0[ph])[half]
            dE += (dl * dl - 2 * dd[None] * dl).sum(dim=1)
        worse = dE[dE > 0].double()
        T_max = float(worse.mean()) / (H * W) ** 2 / np.log(2.0) if worse.numel() else 1.0
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        _, st = lpf.lpf_anneal(pa, d_img[0], -1, target, d_pairs, torch.from_numpy(log_u).cuda(),
                               T_max, 0.01 * T_max, max(1, n // 10), max(1, n // 100))
        dt = time.perf_counter() - t0
        # the paper's own operator: interfacial pixels of different phases, drawn on the device (lpf_anneal_generate)
        d_img2 = torch.from_numpy(start.reshape(H, W).copy()).cuda()
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        _, st2, _ = lpf.lpf_anneal_generate(pa, d_img2, -1, target, lpf.LPF_PROPOSE_INTERFACIAL, inputs.seed_for(7, 3),
                                            torch.from_numpy(log_u).cuda(), T_max, 0.01 * T_max, max(1, n // 10),
                                            max(1, n // 100))
        dt2 = time.perf_counter() - t0
        lpf.lpf_free_paths(pa)
        return {"proposals": n, "seconds": dt, "proposals_per_s": n / dt, "accepted": st["accepted"],
                "E_start": E0, "E_end": st["E"], "levels": st["levels"], "T_max": T_max,
                "interfacial_operator": {"proposals_per_s": n / dt2, "accepted": st2["accepted"], "E_end": st2["E"]}}

    if args.leg:
        out = {"cfg5": measure_swaps, "anneal": measure_anneal, "ensemble": measure_ensemble,
               "s2": lambda: {"cfg2": measure_s2("cfg2"), "cfg3": measure_s2("cfg3")}}[args.leg]()
        print(json.dumps({"leg": args.leg, "result": out}))
        return
    r = measure(w, args.steps, args.warmup, True, strong=(args.scaling == "strong"))
    if args.scaling == "strong" and not r["strong"]:
        args.scaling = "weak"                             # one rank, or a workload with fewer images than ranks
    tests_per_step = lpf_dist.sum_over_ranks(nominal_tests(dict(w, B=r["images_per_gpu"])), device="cuda")
    value = tests_per_step * args.steps / (r["total_ms"] * 1e-3)
    # roofline of the dominant kernel (eval): a UTILISATION of the ALU pipe -- the data operations the design executes
    # at minimum (design_ops, from the uploaded program) over kernel time x derived ALU peak -- and, next to it, of the
    # shared-memory pipe, which binds since the eroded planes (design_smem_bytes over kernel time x 128 B/clk/SM).  The
    # survey's op model (more ops than the design needs) is kept as frac_vs_survey_ops.
    w_loc = dict(w, B=r["images_per_gpu"])               # the eval kernel of THIS rank (strong scaling: its shard)
    d_ops = design_ops(w_loc, r["launch"])
    s_ops = survey_ops(w_loc, r["info"])
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    sm_max_mhz = float(peaks.get("sm_max_mhz", 1965.0))
    peak_ops = SM_COUNT * ALU_LANES_PER_CLK_PER_SM * sm_max_mhz * 1e6
    achieved = d_ops / (r["kernel_ms"] * 1e-3)
    smem_peak = SM_COUNT * 128.0 * sm_max_mhz * 1e6      # 32 banks x 4 B per clock and SM
    smem_rate = design_smem_bytes(w_loc, r["launch"]) / (r["kernel_ms"] * 1e-3)
    measured = lpf.lpf_alu_peak(local_rank) if rank == 0 else None     # live LOP3 / SHF / pair-pattern / POPC rates
    cap = capture_lookup(args.workload, args.flags)                     # ncu --set full of THESE sources, or None
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": r["total_ms"] / args.steps, "higher_is_better": True, "scaling": args.scaling,
        "vs_baseline": None, "dtype": "u32", "data": "synthetic",
        "config": {"workload": args.workload_desc, "images_per_gpu": r["images_per_gpu"], "flags": args.flags or "none",
                   "l2": "flushed with a 256 MiB memset between timed steps",
                   "timing": "sum of per-step CUDA-event times on the launch stream, max over ranks",
                   "launch": r["launch"]},
        "roofline": {"bound": "alu", "achieved": achieved / 1e12, "peak": peak_ops / 1e12, "unit": "T int-op/s",
                     "frac": achieved / peak_ops,
                     "traffic": None if cap is None else cap["dram_read_bytes"] + cap["dram_write_bytes"],
                     "frac_vs_survey_ops": s_ops / (r["kernel_ms"] * 1e-3) / peak_ops,
                     "shared_memory": {"achieved": smem_rate / 1e12, "peak": smem_peak / 1e12, "unit": "TB/s",
                                       "frac": smem_rate / smem_peak,
                                       "how": "row-strip reloads of the uploaded program x (TX + 1) / TX words per start "
                                              "word / kernel time; peak = 148 SM x 128 B/clk x sm_max_mhz"},
                     "ncu": cap, "csrc_sha256": csrc_digest(),
                     "peak_measured": None if measured is None else
                     {"lop3": measured["lop3"] / 1e12, "shf": measured["shf"] / 1e12,
                      "shf_shf_lop3": measured["pair"] / 1e12, "popc": measured["popc"] / 1e12,
                      "unit": "T int-op/s", "how": "lpf_alu_peak: 8 register-only chains per thread, all SMs, live"},
                     "kernel": "eval_kernel", "kernel_ms": r["kernel_ms"], "design_ops_per_launch": d_ops,
                     "survey_ops_per_launch": s_ops,
                     "peak_source": "derived: 148 SM x 64 alu lanes/clk x %.0f MHz (sm_max_mhz of MEASURED_PEAKS.json)"
                                    % sm_max_mhz,
                     "kernel_share_of_step": r["kernel_ms"] * args.steps / r["total_ms"],
                     "note": "frac = data ops the design executes at minimum (per start word: 2 SHF + 1 LOP3 per fused "
                             "pair of program entries, 1 SHF + 1 LOP3 per single entry, POPC + add per terminal; counted "
                             "from the uploaded program) / (kernel time x peak); frac_vs_survey_ops uses SURVEY 8(d)'s "
                             "2 ops per word-node, which the design undercuts, and may exceed 1; shared_memory = the "
                             "same kind of utilisation for the shared-memory pipe (the binding unit: every entry reloads "
                             "a row strip); `ncu` = pipe figures of a committed ncu capture of exactly these sources "
                             "(profiles/capture_index.csv) or null"},
        "e2e": {"value": tests_per_step / r["e2e_s"], "unit": UNIT, "h2d_bytes_per_step": r["e2e"]["h2d"],
                "d2h_bytes_per_step": r["e2e"]["d2h"]},
        "gpu_launches": r["launches_per_step"] * args.steps,
        "clocks": r["clocks"],
    }
    if not args.no_extra and world == 1:
        extra = {}
        for name in sorted(WORKLOADS):
            if name == args.workload:
                continue
            wl = WORKLOADS[name]
            rr = measure(wl, max(3, args.steps // 2), 3, False)
            k = max(3, args.steps // 2)
            cap2 = capture_lookup(name, args.flags)
            extra[name] = {"value": nominal_tests(wl) * k / (rr["total_ms"] * 1e-3), "unit": UNIT,
                           "ms_per_step": rr["total_ms"] / k, "kernel_ms": rr["kernel_ms"],
                           "roofline_frac": design_ops(wl, rr["launch"]) / (rr["kernel_ms"] * 1e-3) / peak_ops,
                           "smem_frac": design_smem_bytes(wl, rr["launch"]) / (rr["kernel_ms"] * 1e-3) / smem_peak,
                           "level": rr["launch"]["level"], "classes": rr["launch"]["classes"],
                           "frac_vs_survey_ops": survey_ops(wl, rr["info"]) / (rr["kernel_ms"] * 1e-3) / peak_ops,
                           "ncu": cap2}
        # the design variants the north star asks to compare, eval kernel alone on the headline workload
        variants = {}
        for vname, vflags, vlevel in (("trie_default", 0, -1), ("trie_level3", 0, 3), ("trie_level2", 0, 2),
                                      ("trie_level1", 0, 1), ("trie_no_e2", lpf.LPF_NO_E2, -1),
                                      ("trie_prune", lpf.LPF_PRUNE, -1), ("one_chain_per_path", lpf.LPF_NO_TRIE, -1)):
            flags_saved, flags = flags, vflags
            variants[vname + "_kernel_ms"] = measure(w, 3, 1, False, level=vlevel)["kernel_ms"]
            flags = flags_saved
        extra["variants_" + args.workload] = variants
        extra["cfg5"] = measure_swaps()
        extra["anneal"] = measure_anneal()
        extra["s2_cfg2"] = measure_s2("cfg2")
        extra["s2_cfg3"] = measure_s2("cfg3")
        extra["ensemble_sum"] = measure_ensemble()
        line["other_workloads"] = extra
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        tests, dt, cores, what = oracle_sample(w, r["imgs"], 20)
        line["cpu_baseline"] = {"value": tests / dt, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": what,
                                "seconds": dt}
        # the paper's CPU column is sequential (one core): the same oracle on one thread, smaller sample
        t1, d1, c1, w1 = oracle_sample(w, r["imgs"], 5, n_vec={2: 800, 3: 200, 4: 2500}[w["cfg"]], threads=1)
        line["cpu_baseline"]["one_thread"] = {"value": t1 / d1, "cores": c1, "sample": w1, "seconds": d1}
    if args.tab1 and rank == 0 and world == 1:
        rows = run_tab1(lpf, torch, local_rank, os.path.join(ROOT, "gpurun_out"))
        line["tab1"] = {"rows": len(rows), "written_to": "gpurun_out/tab1.json, gpurun_out/tab1.md"}
    if args.fig7 and rank == 0 and world == 1:
        rows = run_fig7(lpf, torch, local_rank, os.path.join(ROOT, "gpurun_out"))
        line["fig7"] = {"rows": len(rows), "written_to": "gpurun_out/fig7.json, gpurun_out/fig7.md"}
    if rank == 0:
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
