#!/usr/bin/env python
"""bench.py -- gauge-fix iterations/s and achieved HBM GB/s (BASELINE.json `metric`) on one B200.

A "step" is one pass of the whole hot path = ONE gauge-fixing iteration (K2 fft_xy_fwd, K3
fft_zt_fwd_scale_inv, K4 fft_xy_inv, K5 gbuild_update, K1 delta_theta_F) over one
synthetic lattice.  Default workload: configs[2], 32^4 SU(3), rough links at mean plaquette 0.59 +
Haar gauge transform, alpha = 0.08; headline mode fp64 / 12-real (the paper's best variant,
PAPER.md:72-74), the other three precision x storage modes are reported in "modes".

  python bench.py --gpus N --steps K --warmup W                 # this repo's CUDA path
  python bench.py --impl reference --gpus N --steps K --warmup W  # the oracle on the host cores

The same line carries, under "lattices", the other headline shapes north_star names -- 48^3 x 8
(configs[3]) and 64^4 (configs[4]) -- in all four precision x storage modes (whole-iteration time
from CUDA events around K graph-replayed iterations, per-kernel times from lgf_profile_iterate,
each as a fraction of the measured and of the nominal 8 TB/s HBM roofline); `--lattices none` skips them.

N > 1 (torchrun): "replicas only" -- every rank fixes its own lattice, no data-path collective
(SURVEY.md §8(e)); value = N*K iterations / max-over-ranks device time.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

ALPHA = 0.08
FALLBACK_HBM_GBS = 6650.0          # /opt/skills/guides/B200_PROFILING.md fallback


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=1000)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--lattice", default="32,32,32,32", help="Lx,Ly,Lz,Lt")
    ap.add_argument("--precision", default="f64", choices=["f64", "f32"])
    ap.add_argument("--storage", type=int, default=12, choices=[12, 18])
    ap.add_argument("--modes", default="all", choices=["all", "primary"],
                    help="all: also time the other three precision/storage modes")
    ap.add_argument("--lattices", default="48,48,48,8;64,64,64,64",
                    help="';'-separated extra lattices timed in all four modes under the 'lattices' key ('none' = skip)")
    ap.add_argument("--lattice-steps", type=int, default=20, help="timed iterations per mode on the extra lattices")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--plaquette", type=float, default=0.59)
    return ap.parse_args()


def bytes_per_site(kernel: str, n_l: int, w: int) -> int:
    """Algorithmic bytes per site."""
    if kernel.startswith("K51"):
        return (8 * n_l + 16) * w      # fused update: links read + written once, Delta~ read, Delta written
    if kernel.startswith("K1"):
        return (4 * n_l + 8) * w
    if kernel.startswith("K5"):
        return (8 * n_l + 8) * w
    return 16 * w                      # K2, K3, K4: read + write the 8-real packed Delta


def measured_peak():
    try:
        p = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
        return float(p["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, copy read+write)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md 6.65 TB/s)"


def ncu_traffic(lattice_key: str, mode_key: str, kernel: str):
    """(dram bytes per launch, provenance) of one kernel from the committed `ncu --set full` captures
    (profiles/ncu_traffic.json: dram__bytes_read.sum + dram__bytes_write.sum per launch, with the capture file and the
    commit each figure was taken at), or (None, None) if that kernel / mode / lattice has no capture."""
    try:
        t = json.load(open(os.path.join(ROOT, "profiles", "ncu_traffic.json")))
        e = t.get(lattice_key, {}).get(mode_key, {})
        v = e.get("kernels", {}).get(kernel)
        if v is None:
            return None, None
        return v, {"file": e.get("file"), "commit": e.get("commit"), "metric": "dram__bytes_read.sum + dram__bytes_write.sum per launch"}
    except Exception:
        return None, None


class ClockSampler:
    """nvidia-smi clock / throttle-reason samples every 50 ms, from before the warm-up of the first mode until the last
    timed loop has ended.  The driver's `--steps 20` timed region is only a few milliseconds long, so main() keeps the
    primary mode's iteration loop running (untimed, same kernels) until at least kMinLoadSeconds of load have been sampled."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")
    kMinLoadSeconds = 1.5

    def __init__(self, index: int):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), f"--query-gpu={self.Q}",
                                       "--format=csv,noheader,nounits", "-lms", "50"],
                                      stdout=self.f, stderr=subprocess.DEVNULL)
        except Exception:
            self.p = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": []}
        if self.p is None:
            return out
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except Exception:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        rows, reasons, smax = [], set(), None
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.f.read().splitlines():
            parts = [x.strip() for x in line.split(",")]
            if len(parts) < 7:
                continue
            try:
                rows.append((float(parts[0]), float(parts[2])))
                smax = float(parts[1])
            except ValueError:
                continue
            for n, v in zip(names, parts[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        try:
            os.unlink(self.f.name)
        except OSError:
            pass
        if rows:
            # samples under load: power above the midpoint between the idle floor and the peak of this run
            pw = [r[1] for r in rows]
            thr = min(pw) + 0.5 * (max(pw) - min(pw))
            load = sorted(r[0] for r in rows if r[1] >= thr) or sorted(r[0] for r in rows)
            out["sm_mhz"] = load[len(load) // 2]
            out["samples"] = len(rows)
            out["samples_under_load"] = len(load)
            out["power_w_max"] = max(pw)
        out["sm_max_mhz"] = smax
        out["reasons"] = sorted(reasons)
        return out


def time_oracle(L, U_real, iters: int):
    """The oracle as it stands, timed on the host cores: `iters` iterations (each with its
    measurement) on the given links.  Returns (seconds, threads)."""
    import oracle
    oracle.lib()
    t0 = time.perf_counter()
    oracle.iterate(L, U_real, iters, ALPHA)
    return time.perf_counter() - t0, oracle.threads()


def lattice_name(L) -> str:
    return "x".join(map(str, L))


def workload_name(L, prec: str, stor: int, plaq_target: float) -> str:
    """`config.workload`, the same string in both arms (the reference arm times the fp64 oracle on the same field)."""
    return (f"configs[2]-shaped: {lattice_name(L)} SU(3), {prec}, {stor}-real, rough links plaquette {plaq_target} "
            f"+ Haar gauge transform, alpha {ALPHA}")


def config_dict(L, prec: str, stor: int, plaq_target: float, plaq: float, world: int, peak: float, peak_src: str) -> dict:
    """`config` of the JSON line -- the SAME dictionary in the CUDA arm and in the reference arm (the oracle computes in
    fp64 on full 3x3 links whatever `prec` / `stor` say: they name the workload the ratio is taken on)."""
    V = L[0] * L[1] * L[2] * L[3]
    w = 8 if prec == "f64" else 4
    return {"workload": workload_name(L, prec, stor, plaq_target), "measured_plaquette": round(plaq, 6), "sites": V,
            "parallelism": "replicas only" if world > 1 else "1 GPU",
            "l2": ("inputs larger than L2 (links %.0f MB > 126 MB)" if 4 * stor * V * w > 126e6 else
                   "L2-resident workload (links %.0f MB): launch-bound, reported without a roofline claim") % (4 * stor * V * w / 1e6),
            "hbm_peak_GBps": peak, "hbm_peak_source": peak_src}


def run_reference(args, L):
    """--impl reference: the oracle (unmodified, as it stands) on the box's host cores, same config / metric / unit as
    the CUDA arm; each step = one full oracle iteration of the same lattice (about 1 s at 32^4 on 16 threads), W warm-up
    and K timed steps as asked, capped at 60 iterations in total so that the run ends within a few minutes."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import torch
    import lgf_inputs as gi
    V = gi.volume(L)
    dev = "cuda" if torch.cuda.is_available() else "cpu"
    U = gi.make_config(L, gi.CONFIG_SEED + 2, args.plaquette, device=dev)
    plaq = gi.mean_plaquette(U, L)
    U = U.cpu()
    Ur = gi.as_real(U)
    peak, peak_src = measured_peak()
    per_iter_cap = 60 if V <= (1 << 20) else 4
    steps = max(1, min(args.steps, per_iter_cap))
    warm = max(0, min(args.warmup, per_iter_cap - steps, 5))
    if warm:
        time_oracle(L, Ur, warm)
    sec, thr = time_oracle(L, Ur, steps)
    # oracle.iterate does 1 initial measurement + steps x (update + measurement)
    val = steps / sec
    line = {
        "impl": "reference", "metric": "gauge_fix_iterations_per_s", "value": val, "unit": "iterations/s",
        "n_gpus": args.gpus, "steps": steps, "warmup": warm, "ms_per_step": 1e3 * sec / steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": config_dict(L, args.precision, args.storage, args.plaquette, plaq, 1, peak, peak_src),
        "note": "oracle/lgf_oracle.cpp (plain C++, fp64, full 3x3 links, OpenMP over sites/lines) on host cores",
        "cpu_baseline": {"value": val, "unit": "iterations/s", "cores": thr, "kind": "oracle",
                         "sample": f"{steps} full iterations of the {lattice_name(L)} lattice"},
        "e2e": {"value": val, "unit": "iterations/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


ALL_MODES = [("f64", 18), ("f64", 12), ("f32", 18), ("f32", 12)]


def main():
    args = parse_args()
    L = tuple(int(x) for x in args.lattice.split(","))
    if args.impl == "reference":
        run_reference(args, L)
        return

    import torch
    import torch.distributed as dist
    import lgf_inputs as gi
    import paper_1208_1186_b200 as lgf
    from paper_1208_1186_b200 import replicas

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the lgf library has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    K, W = args.steps, max(args.warmup, 3)
    peak, peak_src = measured_peak()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def time_modes(Lx, U, modes, K_, W_, hold_primary_s=0.0):
        """Time K_ graph-replayed iterations (after W_ warm-up iterations) of lattice Lx in every mode of `modes`, then the
        per-kernel split.  Inputs are resident in HBM before the timed region.  Returns {(prec, stor): result}."""
        Vx = gi.volume(Lx)
        lkey = lattice_name(Lx)
        out = {}
        for i, (prec, stor) in enumerate(modes):
            dt = torch.float64 if prec == "f64" else torch.float32
            gf = lgf.GaugeFixer(Lx, lgf.LGF_F64 if prec == "f64" else lgf.LGF_F32, stor, device=str(dev))
            Ud = gi.as_real(U, dt)                       # device tensor: inputs resident in HBM
            gf.load(Ud)
            del Ud
            gf.iterate(W_, ALPHA)                        # warm-up (also captures the graph)
            stream = torch.cuda.current_stream(dev)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            barrier()
            n0 = gf.launch_count()
            e0.record(stream)
            gf.iterate_async(K_, ALPHA)
            e1.record(stream)
            res = gf.wait()
            barrier()
            launches = gf.launch_count() - n0
            ms = replicas.max_over_ranks(e0.elapsed_time(e1), dev)
            kern_ms, _ = gf.profile_iterate(20, ALPHA)
            if i == 0 and hold_primary_s > 0:
                # keep the same kernels running (untimed, after both measurements) so that the 50 ms clock sampler sees
                # them under load; a second of fp64 iterations drives the board into its 1 kW power cap (sw_power_cap),
                # which the short timed region above does not reach
                t_end = time.perf_counter() + hold_primary_s
                while time.perf_counter() < t_end:
                    gf.iterate(max(K_, 50), ALPHA)
            info = gf.path_info()
            w = 8 if prec == "f64" else 4
            b_iter = (12 * stor + 64) * w
            kernels = {}
            for k, t_ms in kern_ms.items():
                b = bytes_per_site(k, stor, w) * Vx
                frac = b / (t_ms * 1e-3) / 1e9 / peak
                kernels[k] = {"ms": t_ms, "algorithmic_GBps": b / (t_ms * 1e-3) / 1e9, "frac_of_peak": frac,
                              "share_of_iteration": t_ms / sum(kern_ms.values())}
                dram, src = ncu_traffic(lkey, f"{prec}_{stor}", k)
                if dram is not None:
                    # what the kernel really pulled through HBM under ncu (cold L2) over the live time: an upper bound of
                    # its HBM rate inside the pipeline, where Delta-sized fields may be L2-resident (SURVEY.md §8(d) caveat)
                    kernels[k]["ncu_dram_bytes"] = dram
                    kernels[k]["ncu_dram_GBps"] = dram / (t_ms * 1e-3) / 1e9
                    kernels[k]["ncu_source"] = src
                if frac > 1.0:
                    kernels[k]["note"] = "above the copy peak: part of this kernel's algorithmic bytes are served by the L2"
            out[(prec, stor)] = {
                "iterations_per_s": world * K_ / (ms * 1e-3), "ms_per_iteration": ms / K_,
                "site_updates_per_s": world * K_ * Vx / (ms * 1e-3),
                "algorithmic_GBps": b_iter * Vx * K_ / (ms * 1e-3) / 1e9,
                "frac_of_hbm_peak": b_iter * Vx * K_ / (ms * 1e-3) / 1e9 / peak,
                "frac_of_nominal_8TBps": b_iter * Vx * K_ / (ms * 1e-3) / 1e9 / 8000.0,   # north_star's nominal figure
                "bytes_per_site_iteration": b_iter, "theta": res.theta, "F": res.F, "steps": K_,
                "launches": launches, "fft_path": info["fft_path"], "fused_update": info["fused"],
                "kernels_below_0.70_of_peak": sorted(k for k, v in kernels.items() if v["frac_of_peak"] < 0.70),
                "kernels": kernels,
            }
            gf.close()
            del gf
            torch.cuda.empty_cache()
        return out

    # every rank: its own seeded lattice (replicas only)
    V = gi.volume(L)
    U = gi.make_config(L, replicas.rank_seed(gi.CONFIG_SEED + 2, rank), args.plaquette, device=dev)
    plaq = gi.mean_plaquette(U, L)
    primary = (args.precision, args.storage)
    modes = [primary] + ([m for m in ALL_MODES if m != primary] if args.modes == "all" else [])

    sampler = ClockSampler(local) if rank == 0 else None
    t_load0 = time.perf_counter()
    results = time_modes(L, U, modes, K, W, hold_primary_s=ClockSampler.kMinLoadSeconds if rank == 0 or world > 1 else 0.0)
    total_launches = results[primary]["launches"]

    # ---- e2e: the user's call sequence with HOST buffers: load (H2D) + fix/iterate + store (D2H) ----
    e2e = None
    if not args.no_e2e:
        prec, stor = primary
        dt = torch.float64 if prec == "f64" else torch.float32
        host_in = gi.as_real(U, dt).cpu().pin_memory()
        host_out = torch.empty_like(host_in).pin_memory()
        gf = lgf.GaugeFixer(L, lgf.LGF_F64 if prec == "f64" else lgf.LGF_F32, stor, device=str(dev))
        # untimed warm-up of the same three calls (first launches load their kernels lazily)
        gf.load(host_in)
        gf.iterate(W, ALPHA)
        gf.fix(ALPHA, 1e-15, W)
        gf.store(host_out)
        barrier()
        t0 = time.perf_counter()
        gf.load(host_in)
        if prec == "f64":
            r = gf.fix(ALPHA, 1e-15, 5000)
        else:
            r = gf.iterate(50, ALPHA)
        gf.store(host_out)
        torch.cuda.synchronize()
        sec = time.perf_counter() - t0
        sec = replicas.max_over_ranks(sec, dev)
        nb = host_in.numel() * host_in.element_size()
        e2e = {"value": world * r.iterations / sec, "unit": "iterations/s",
               "h2d_bytes_per_step": nb / max(r.iterations, 1), "d2h_bytes_per_step": nb / max(r.iterations, 1),
               "job": f"lgf_load(host pinned) + {'lgf_fix(theta<1e-15)' if prec == 'f64' else 'lgf_iterate(50)'} + lgf_store(host)",
               "iterations": r.iterations, "seconds": sec, "theta": r.theta, "F": r.F,
               "h2d_bytes": nb, "d2h_bytes": nb}
        gf.close()
        del gf, host_in, host_out

    # ---- the other headline lattices (configs[3], configs[4]); rank 0's clocks keep being sampled ----
    lattices = {}
    if args.lattices != "none":
        for spec in args.lattices.split(";"):
            Lx = tuple(int(x) for x in spec.split(","))
            if Lx == L:
                continue
            idx = 3 if Lx == (48, 48, 48, 8) else 4
            Ux = gi.make_config(Lx, replicas.rank_seed(gi.CONFIG_SEED + idx, rank), 0.58 if idx == 3 else 0.59, device=dev)
            rx = time_modes(Lx, Ux, ALL_MODES, args.lattice_steps, 3)
            del Ux
            torch.cuda.empty_cache()
            lattices[lattice_name(Lx)] = {"sites": gi.volume(Lx), "steps": args.lattice_steps, "warmup": 3,
                                          "modes": {f"{p}_{s}": r for (p, s), r in rx.items()}}
    clocks = sampler.stop() if sampler else None

    # ---- launch-bound lattices: one at a time and batched per launch (lgf_create_batch) ----
    small = {}
    if args.lattices != "none" and rank == 0:
        for Ls, nb in (((8, 8, 8, 8), 64), ((16, 16, 16, 16), 16)):
            ent = {}
            for B in (1, nb):
                Ub = torch.cat([gi.as_real(gi.make_config(Ls, gi.CONFIG_SEED + 10 + b, 0.59, device=dev)) for b in range(B)], 0)
                gf = lgf.GaugeFixer(Ls, lgf.LGF_F64, 12, device=str(dev), nbatch=B)
                gf.load(Ub)
                gf.iterate(20, ALPHA)
                stream = torch.cuda.current_stream(dev)
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                torch.cuda.synchronize()
                e0.record(stream)
                gf.iterate_async(200, ALPHA)
                e1.record(stream)
                gf.wait()
                torch.cuda.synchronize()
                us = e0.elapsed_time(e1) * 1e3 / 200
                ent["single" if B == 1 else f"batch_{B}"] = {
                    "us_per_launch_set": us, "us_per_lattice_iteration": us / B, "lattice_iterations_per_s": B / (us * 1e-6),
                    "path": "one 16-CTA cluster per lattice (k_cluster8_iterate)" if "k_cluster8_iterate" in gf.describe() else "launch graph"}
                gf.close()
                del gf, Ub
            small[lattice_name(Ls) + " f64_12"] = ent

    # ---- CPU baseline: the oracle, bounded sample, rank 0 at N = 1 only ----
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        iters = 3 if V <= (1 << 20) else 1
        sec, thr = time_oracle(L, gi.as_real(U).cpu(), iters)
        cpu = {"value": iters / sec, "unit": "iterations/s", "cores": thr, "kind": "oracle",
               "sample": f"{iters} full iterations of the same {lattice_name(L)} lattice ({sec:.1f} s)"}

    if rank == 0:
        pr = results[primary]
        dom = max(pr["kernels"].items(), key=lambda kv: kv[1]["ms"])
        w = 8 if primary[0] == "f64" else 4
        dom_bytes = bytes_per_site(dom[0], primary[1], w) * V
        traffic, traffic_src = ncu_traffic(lattice_name(L), f"{primary[0]}_{primary[1]}", dom[0])
        line = {
            "metric": "gauge_fix_iterations_per_s", "value": pr["iterations_per_s"], "unit": "iterations/s",
            "n_gpus": world, "steps": K, "warmup": W, "ms_per_step": pr["ms_per_iteration"],
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": primary[0], "data": "synthetic",
            "config": config_dict(L, primary[0], primary[1], args.plaquette, plaq, world, peak, peak_src),
            "site_updates_per_s": pr["site_updates_per_s"],
            "achieved_HBM_GBps_algorithmic": pr["algorithmic_GBps"],
            "iteration_frac_of_hbm_roofline": pr["frac_of_hbm_peak"],
            "iteration_frac_of_nominal_8TBps": pr["frac_of_nominal_8TBps"],
            "roofline": {"bound": "hbm", "kernel": dom[0], "achieved": dom[1]["algorithmic_GBps"], "peak": peak,
                         "unit": "GB/s", "frac": dom[1]["frac_of_peak"], "traffic": traffic, "traffic_source": traffic_src,
                         "algorithmic_bytes_per_launch": dom_bytes, "peak_source": peak_src},
            "cpu_baseline": cpu,
            "e2e": e2e,
            "gpu_launches": total_launches,
            "clocks": clocks,
            "modes": {f"{p}_{s}": {k: v for k, v in r.items()} for (p, s), r in results.items()},
            "lattices": lattices,
            "small_lattices": small,
        }
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
