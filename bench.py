"""bench.py — throughput of the SPIIR hot path on B200 (one JSON line on stdout).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N ... bench.py --gpus N ...

A *step* is one pass of the whole hot path over one 1-second chunk of synthetic strain
(DESIGN.md §8): spiir_filter_chunk (decimator chain, IIR recursion, band sums, up-sample
cascade, SNR ring, fused per-template maximum) -> spiir_peaks (threshold 4, mode 0) ->
coherent_sky_search on the previous chunk's candidates (one-chunk lag, reading A13) ->
timeslide_background with 100 slides of 1 s.  Workload at N = 1: BASELINE.json config 4
(H1/L1/V1, 20 000 templates x 700 filters over 8 rate bands, HEALPix nside 32, 100
slides), synthetic and seeded (workloads/).  N > 1: every rank runs one such template
shard (weak scaling; the path has no exchange step).

`value` = filter-sample updates/s of the whole job, all stages inside the timed region,
inputs resident in HBM; `e2e` = the same through the C ABI with pinned HOST strain in and
HOST candidate / result arrays out.  `--impl reference` times the float64 oracle (oracle/)
on the host cores on a bounded sample of the same workload.
"""
import argparse
import json
import math
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

METRIC = "spiir_filter_sample_updates_per_s"
UNIT = "updates/s"
FLOP_PER_UPDATE = 12.0          # 12 flop per filter-sample (8 FP32 instructions)
FLOP_PER_EVAL = 9.0             # EXECUTED by k_sky per direction (N_d = 3): 1 FMUL + 4 FFMA, the five-term quadratic form of
                                # Eq. 28 (the |z_T|^2 term is a constant: the projector has trace 2).  One basis for
                                # roofline.frac: executed work.  Other countings of the same evaluation, as context only:
FLOP_PER_EVAL_CONTEXT = {"paper_4_Nd_squared": 36.0,
                         "survey_fp32_instructions": 22.0,     # SURVEY.md section 8(d), the direct two-projection form
                         "six_term_quadratic_form_round1": 11.0}
# FP32 ALU roofline: 148 SMs x 128 FP32 lanes x 2 flop (FMA) x 1.965 GHz (B200_PROFILING.md
# unit counts and clocks.max.sm).  The recursion's instruction mix (2 FMUL + 4 FFMA + 2 FADD = 12 flop in
# 8 issue slots) tops out at 12/16 = 75 % of it.
FP32_PEAK_TFLOPS = 148 * 128 * 2 * 1.965e9 / 1e12
FP32_LANE_OPS_PER_S = 148 * 128 * 1.965e9


def ncu_traffic_bytes():
    """dram__bytes_read.sum + dram__bytes_write.sum of the two hot kernels, summed over the launches of ONE step,
    read from the committed `ncu --set full` export profiles/r2_traffic.csv (kernel, launches per step, bytes);
    None for a kernel without a capture.  The number is a record of that capture, not measured by this run."""
    out = {"k_bank": None, "k_sky": None}
    path = os.path.join(ROOT, "profiles", "r2_traffic.csv")
    try:
        for line in open(path):
            f = [x.strip() for x in line.split(",")]
            if len(f) >= 3 and f[0] in out:
                out[f[0]] = float(f[2])
    except OSError:
        pass
    return out


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=4, help="BASELINE.json config index (1, 2 or 4 stream a bank; 3 = sky search alone)")
    ap.add_argument("--templates", type=int, default=None, help="override the template count (debugging)")
    ap.add_argument("--slides", type=int, default=None, help="override the number of time slides")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-cfg3", action="store_true", help="skip the config-3 sky-search row (about 15 s of set-up)")
    ap.add_argument("--no-parity", action="store_true", help="skip the sampled oracle check after the timed region")
    ap.add_argument("--fast-norm", action="store_true",
                    help="diagonal approximation of the bank's noise normalisation (quicker set-up)")
    return ap.parse_args()


# ----------------------------------------------------------------------------- clocks
class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms DURING the timed region."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index):
        self.rows, self.proc, self.thr = [], None, None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(gpu_index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thr = threading.Thread(target=self._read, daemon=True)
            self.thr.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def stop(self, t0, t1):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons, pw = [], [], set(), []
        for ts, line in self.rows:
            f = [x.strip() for x in line.split(",")]
            if len(f) < 9:
                continue
            inside = t0 - 0.1 <= ts <= t1 + 0.3
            try:
                if inside:
                    sm.append(float(f[1])); pw.append(float(f[3]))
                mx.append(float(f[2]))
            except ValueError:
                continue
            if inside:
                for name, val in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"),
                                     f[5:9]):
                    if val.lower().startswith("active"):
                        reasons.add(name)
        if not sm:                                   # timed region shorter than one sample: take all samples
            for ts, line in self.rows:
                f = [x.strip() for x in line.split(",")]
                try:
                    sm.append(float(f[1]))
                except (ValueError, IndexError):
                    pass
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


# ----------------------------------------------------------------------------- workload
def workload_params(args):
    import workloads
    cfg = workloads.config(args.config)
    if not cfg["n_templates"]:
        raise SystemExit("config %d has no filter bank; bench streams configs 1, 2 or 4" % args.config)
    T = args.templates or cfg["n_templates"]
    S = cfg["n_slides"] if args.slides is None else args.slides
    f_in = cfg["band_rates"][0]
    return dict(cfg=cfg, T=T, S=S, D=len(cfg["dets"]), chunk=f_in, n_out=2048, nside=cfg["nside"],
                n_pix=12 * cfg["nside"] ** 2, ring_len=(S + 3) * 2048, thr=float(cfg["threshold"]))


def updates_per_chunk(bank, D, chunk):
    """Filter-sample updates of one chunk: every filter advances (chunk >> band) samples, per detector."""
    band = np.asarray(bank["band"]).astype(np.int64)
    return int(D * np.sum(chunk >> band))


# ----------------------------------------------------------------------------- oracle sample (CPU)
_SAMPLE_INPUTS = {}
# Fraction of (detector, template, second) slots above SNR 4 in steady state, as the CUDA arm measures it on config 4
# (~40 500 candidates of 60 000 slots per chunk, BENCH_r01 / r02; tests/test_gpu_parity.py::test_cfg4_steady_state);
# used only when the sampled seconds are still in the bank's cold-start transient and show none.
STEADY_TRIGGER_FRACTION = 0.675


def oracle_setup():
    """The timed build of the oracle (-O3 -march=native -fopenmp, compiled on this box)
    on the physical cores.  Returns the thread count."""
    import oracle
    return oracle.use_timed_build()


def oracle_sample(args, n_templates, n_chunks, n_trig, repeat=1, threads=None):
    """Times the float64 oracle (oracle/, as it stands) on a bounded sample of the workload:
    the first `n_templates` templates over `n_chunks` seconds (O1-O4) and the sky search with
    all its slides for `n_trig` candidates on packed SNR snippets (O6-O7).  Work is linear in
    templates and in candidates, so rates extrapolate to the full chunk."""
    import oracle
    import workloads
    w = workload_params(args)
    cfg, D, S = w["cfg"], w["D"], w["S"]
    key = (args.config, n_templates, n_chunks)
    if key not in _SAMPLE_INPUTS:                      # inputs are generated once, outside the timed calls
        _SAMPLE_INPUTS[key] = (workloads.bank_for_config(args.config, n_templates=n_templates),
                               workloads.strain_for_config(args.config, seconds=n_chunks)["strain"])
    bank, x = _SAMPLE_INPUTS[key]
    if threads:
        oracle.set_threads(threads)
    dec, itp = workloads.halfband_taps()
    multirate = len(cfg["band_rates"]) > 1
    out = dict(threads=oracle.num_threads(), n_templates=n_templates, n_chunks=n_chunks, n_trig=n_trig)
    t_bank = t_peaks = t_sky = 0.0
    for _ in range(repeat):
        t0 = time.perf_counter()
        z = oracle.filter_bank(x, bank, dec if multirate else None, itp if multirate else None)
        t1 = time.perf_counter()
        n_valid = 0
        for c in range(n_chunks):
            zc = np.ascontiguousarray(z[:, :, c * 2048:(c + 1) * 2048]).reshape(D * n_templates, 2048)
            _, v = oracle.peaks_mode0(zc, w["thr"])
            n_valid += int(v.sum())
        t2 = time.perf_counter()
        t_bank += t1 - t0
        t_peaks += t2 - t1
    out["updates"] = updates_per_chunk(bank, D, w["chunk"]) * n_chunks * repeat
    out["t_bank"], out["t_peaks"] = t_bank, t_peaks
    out["trigger_fraction"] = n_valid / float(D * n_templates * n_chunks)
    out["evals"], out["t_sky"] = 0, 0.0
    if w["nside"] and n_trig:
        pos, resp = workloads.detector_geometry(cfg["dets"])
        U2, delay = oracle.sky_table(w["nside"], pos, resp, cfg["sigma"], 1.234, 2048.0)
        u2 = U2.astype(np.float32)
        half = 102
        W = 2 * half + 1
        rng = np.random.default_rng(cfg["seed"])
        zs, tdet, k, _ = workloads.snr_snippets(rng, u2, delay, n_trig, S + 1, half, 0.1)
        zc = np.ascontiguousarray(zs).view(np.complex64)[..., 0]
        L = zc.shape[2]
        ones, rows = np.ones(n_trig, np.int32), np.arange(n_trig, dtype=np.int32)
        for _ in range(repeat):
            t0 = time.perf_counter()
            oracle.sky_search(u2, delay, zc, n_trig * L, L, L, L - 1, ones, rows, tdet, k)
            if S:
                oracle.sky_search(u2, delay, zc, n_trig * L, L, L, L - 1, ones, rows, tdet, k,
                                  n_slides=S, step=W, slide_mult=[1] * D)
            t_sky += time.perf_counter() - t0
        out["evals"] = n_trig * w["n_pix"] * (1 + S) * repeat
        out["t_sky"] = t_sky
    return out


def oracle_whole_step_rate(s, updates_full, evals_full, slots_full):
    """Whole-path updates/s of the oracle extrapolated to one full chunk from the sampled stage rates."""
    t = updates_full / (s["updates"] / s["t_bank"])
    t += s["t_peaks"] * slots_full / float(max(1, s["n_templates"] * s["n_chunks"]))
    if s["evals"]:
        t += evals_full / (s["evals"] / s["t_sky"])
    return updates_full / t, t


def cpu_leg(args, w, n_t, n_c, n_trig, steps=1, warmup=0):
    """The oracle on the host cores: `steps` timed repetitions of one bounded sample after `warmup` untimed
    ones, on all physical cores, plus one single-thread pass over an eighth of the sample.  Both CPU legs of
    this file (--impl reference and cpu_baseline) go through here, with samples that fill the cores."""
    import oracle
    import workloads
    threads = oracle_setup()
    for _ in range(max(0, warmup)):
        oracle_sample(args, n_t, n_c, n_trig, threads=threads)
    acc = None
    t0 = time.perf_counter()
    for _ in range(max(1, steps)):
        s = oracle_sample(args, n_t, n_c, n_trig, threads=threads)
        if acc is None:
            acc = dict(s)
        else:
            for key in ("updates", "t_bank", "t_peaks", "evals", "t_sky"):
                acc[key] += s[key]
    wall = time.perf_counter() - t0
    one = oracle_sample(args, max(16, n_t // 8), n_c, max(4, n_trig // 8) if n_trig else 0, threads=1)
    oracle.set_threads(threads)
    per_t = updates_per_chunk(workloads.bank_for_config(args.config, n_templates=min(n_t, 64)), w["D"], w["chunk"]) / min(n_t, 64)
    updates_full = per_t * w["T"]
    slots_full = w["D"] * w["T"]
    frac = acc["trigger_fraction"] if acc["trigger_fraction"] > 0.05 else STEADY_TRIGGER_FRACTION
    return dict(acc=acc, wall=wall, threads=threads, one=one, updates_full=updates_full, slots_full=slots_full,
                trigger_fraction=frac)


def cpu_baseline_dict(leg, value, t_chunk, w, S):
    acc, one = leg["acc"], leg["one"]
    import multiprocessing
    return {
        "value": value, "unit": UNIT, "cores": leg["threads"], "logical_cpus": multiprocessing.cpu_count(),
        "kind": "oracle", "build": "gcc -O3 -march=native -fopenmp -ffp-contract=off (compiled on this box)",
        "bank_updates_per_s": acc["updates"] / acc["t_bank"],
        "sky_evals_per_s": (acc["evals"] / acc["t_sky"]) if acc["evals"] else None,
        "single_thread": {"bank_updates_per_s": one["updates"] / one["t_bank"],
                          "sky_evals_per_s": (one["evals"] / one["t_sky"]) if one["evals"] else None},
        "extrapolated_s_per_chunk": t_chunk,
        "sample": "per repetition: first %d templates x %d s through O1-O4 (%.2f s in all) and %d candidates x %d "
                  "directions x (1+%d slides) through O6-O7 (%.2f s in all); whole-chunk rate extrapolated linearly in "
                  "templates and candidates" % (acc["n_templates"], acc["n_chunks"], acc["t_bank"], acc["n_trig"],
                                                w["n_pix"], S, acc["t_sky"])}


def run_reference(args):
    """--impl reference: the oracle on the host cores, K timed steps after W warm-ups; each step is one bounded
    sample that fills the cores (1024 templates x 1 s through O1-O4, 16 candidates per thread through O6-O7)."""
    w = workload_params(args)
    import oracle
    from oracle.build import physical_cores
    n_t, n_c = min(1024, w["T"]), 1
    n_trig = max(256, 16 * physical_cores()) if w["nside"] else 0
    leg = cpu_leg(args, w, n_t, n_c, n_trig, steps=args.steps, warmup=args.warmup)
    acc = leg["acc"]
    evals_full = leg["trigger_fraction"] * leg["slots_full"] * w["n_pix"] * (1 + w["S"]) if w["nside"] else 0
    value, t_chunk = oracle_whole_step_rate(acc, leg["updates_full"], evals_full, leg["slots_full"])
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * leg["wall"] / max(1, args.steps),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": config_dict(args, w),
        "bank_updates_per_s": acc["updates"] / acc["t_bank"],
        "sky_evals_per_s": (acc["evals"] / acc["t_sky"]) if acc["evals"] else None,
        "extrapolated_s_per_chunk": t_chunk,
        "cpu_baseline": cpu_baseline_dict(leg, value, t_chunk, w, w["S"]),
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def config_dict(args, w):
    cfg = w["cfg"]
    return {"workload": "BASELINE.json configs[%d] (%s): %d det, %d templates x %d filters, %d rate bands, "
                        "1-s chunks of %d samples, peaks mode 0 thr %.1f, HEALPix nside %d, %d time slides of 1 s"
                        % (args.config, cfg["name"], w["D"], w["T"], cfg["filters_per_template"],
                           len(cfg["band_rates"]), w["chunk"], w["thr"], w["nside"], w["S"]),
            "templates_per_gpu": w["T"], "ring_seconds": w["ring_len"] // 2048,
            "l2": "no flush: per-step working set (coefficients, states, band sums, SNR ring segment) exceeds the 126 MB L2",
            "parallelism": "template shards, no collective"}


def parity_check(args, w, bank, x, fed, bk, prev_trig, fg_out, bg_out, u2, delay, mult, dec, itp, n_tmpl=8):
    """Sampled oracle check of the run that was just timed (same process, same device state)."""
    import torch
    import oracle
    import paper_2011_06787_b200 as sp
    D, T, S, chunk = w["D"], w["T"], w["S"], w["chunk"]
    n_slots = D * T
    view = bk.snr_view()
    L, k_new = int(view.c.ring_len), int(view.c.k_newest)
    tp = sp.triggers_to_numpy(prev_trig)
    rng = np.random.default_rng(w["cfg"]["seed"] + 99)
    have = np.unique(tp["tmpl"][tp["valid"] == 1])
    if have.size == 0:
        return {"n": 0, "note": "no candidate in the last step"}
    sel = np.unique(np.concatenate([have[:2], rng.choice(have, size=min(n_tmpl - 2, have.size), replace=False)]))[:n_tmpl]
    # (1) SNR end to end: the oracle over every chunk fed so far, for the sampled templates
    xs = np.concatenate([x[:, c * chunk:(c + 1) * chunk] for c in fed], axis=1)
    z_ref = oracle.filter_bank(xs, bank, dec, itp, templates=sel.astype(np.int64))       # [D][n_sel][n_fed * 2048]
    rows = bk.ring_rows(torch.from_numpy(sel.astype(np.int64)).cuda())                    # [D][n_sel][L][2] float32
    zr = rows.cpu().numpy().view(np.complex64)[..., 0]                                    # ring index = k mod L
    n_out = z_ref.shape[2]
    assert n_out == k_new + 1, (n_out, k_new)
    kk = np.arange(max(0, n_out - L), n_out)
    err_snr = float(np.abs(zr[:, :, kk % L].astype(np.complex128) - z_ref[:, :, kk]).max())
    # (2) the sky results of the sampled templates' candidates against O6 / O7 on the GPU's ring
    slot_rows = (np.arange(D)[:, None] * T + sel[None, :]).reshape(-1)
    sub = tp[slot_rows].copy()
    sub["tmpl"] = np.tile(np.arange(len(sel)), D)
    fg = sp.results_to_numpy(fg_out)[slot_rows]
    bg = sp.results_to_numpy(bg_out).reshape(n_slots, max(S, 1))[slot_rows] if S else None
    worst, n_res, bad_pix = 0.0, 0, 0
    for res, kw in ((fg.reshape(-1, 1), {}), (bg, dict(n_slides=S, step=2048, slide_mult=mult))):
        if res is None:
            continue
        out, pix, _ = oracle.sky_search(u2, delay, zr, len(sel) * L, L, L, k_new, sub["valid"], sub["tmpl"],
                                        sub["det"], sub["k"], **kw)
        has = pix >= 0
        if not np.array_equal(res["pix"] >= 0, has):
            bad_pix += int(((res["pix"] >= 0) != has).sum())
            continue
        c = out[..., 0]
        rel = np.abs(res["coh2"].astype(np.float64) - c)[has] / np.maximum(c[has], 1e-30)
        worst = max(worst, float(rel.max()) if rel.size else 0.0)
        n_res += int(has.sum())
        for i, sl in np.argwhere(has & (res["pix"] != pix)):
            ok, cc, _, _ = oracle.sky_eval(u2, delay, zr, len(sel) * L, L, L, k_new, int(sub["tmpl"][i]), int(sub["det"][i]),
                                           int(sub["k"][i]), int(res["pix"][i, sl]), s=(sl + 1 if kw else 0),
                                           step=2048 if kw else 0, slide_mult=mult if kw else None)
            if not (ok and cc >= c[i, sl] - max(1e-4 * c[i, sl], 1e-3)):
                bad_pix += 1
    ok = err_snr <= 1e-3 and worst <= 1e-4 and bad_pix == 0
    return {"ok": bool(ok), "templates": int(len(sel)), "chunks_streamed": len(fed), "ring_wrapped": bool(k_new + 1 > L),
            "snr_samples": int(zr[:, :, kk % L].size), "max_abs_err_snr": err_snr, "tol_snr": 1e-3,
            "sky_results": n_res, "max_rel_err_coh2": worst, "tol_coh2_rel": 1e-4, "pixels_not_argmax": bad_pix,
            "n": int(zr[:, :, kk % L].size) + n_res, "max_err": max(err_snr, worst)}


# ----------------------------------------------------------------------------- the CUDA arm
def run_ours(args):
    import torch
    import torch.distributed as dist
    import workloads
    import paper_2011_06787_b200 as sp
    from paper_2011_06787_b200 import shard as shd

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback; --impl reference times the oracle)")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    sp.lib()                                             # fails loudly if libspiir_b200.so is missing

    if args.config == 3:
        # the sky-search stress config has no filter bank: one line with the sky search alone (single GPU; the default
        # line carries the same row as `sky_stress_cfg3`)
        if rank == 0:
            row = sky_stress_cfg3_row(sp, workloads, torch, reps=max(1, args.steps))
            ms = row["ms_foreground"] + row["ms_slides"]
            print(json.dumps({"metric": "spiir_sky_evals_per_s", "value": row["evals_per_s"], "unit": "evals/s", "n_gpus": 1,
                              "steps": max(1, args.steps), "warmup": 1, "ms_per_step": ms, "higher_is_better": True,
                              "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                              "config": {"workload": row["workload"], "l2": "no flush: 2 GB of snippets per pass"},
                              "roofline": {"kernel": "k_sky", "bound": "alu", "achieved": FLOP_PER_EVAL * row["evals_per_s"] / 1e12,
                                           "peak": FP32_PEAK_TFLOPS, "unit": "TFLOP/s", "frac": row["frac_of_fp32_peak"],
                                           "traffic": None, "flop_per_unit": "9 executed per evaluation"},
                              "sky_stress_cfg3": row}), flush=True)
        if world > 1:
            dist.destroy_process_group()
        return
    w = workload_params(args)
    cfg, T, S, D, chunk = w["cfg"], w["T"], w["S"], w["D"], w["chunk"]
    multirate = len(cfg["band_rates"]) > 1
    t_setup = time.time()
    bank = workloads.bank_for_config(args.config, n_templates=T, exact_norm=not args.fast_norm, shard=rank)
    st = workloads.strain_for_config(args.config)
    x = st["strain"]
    n_chunks = x.shape[1] // chunk
    dec, itp = workloads.halfband_taps()
    upd_chunk = updates_per_chunk(bank, D, chunk)
    n_slots = D * T
    has_sky = w["nside"] > 0

    bk = sp.Bank(bank, D, chunk, ring_len=w["ring_len"], bank_size=1000,
                 dec_taps=dec if multirate else None, int_taps=itp if multirate else None)
    assert bk.updates_per_chunk(chunk) == upd_chunk
    plan = None
    if has_sky:
        pos, resp = workloads.detector_geometry(cfg["dets"])
        u2, delay = sp.sky_table_build(w["nside"], pos, resp, cfg["sigma"], st["gmst"], 2048.0)
        plan = sp.SkyPlan(u2, delay, max_slots=n_slots)
    mult = [1] * D
    # strain chunks: [n_chunks][D][chunk], resident in HBM and as pinned host memory
    xc = np.ascontiguousarray(x.reshape(D, n_chunks, chunk).transpose(1, 0, 2))
    x_host = torch.from_numpy(xc).pin_memory()
    x_dev = x_host.to(dev)
    x_in = torch.empty(D, chunk, dtype=torch.float32, device=dev)        # e2e staging buffer
    trig = [torch.zeros(n_slots, 40, dtype=torch.uint8, device=dev) for _ in range(2)]
    max_steps = w["ring_len"] // 2048 + 2 * (args.warmup + args.steps) + 8
    counts = torch.zeros(max_steps, dtype=torch.int32, device=dev)
    fg_out = torch.zeros(n_slots, 16, dtype=torch.uint8, device=dev)
    bg_out = torch.zeros(n_slots * max(S, 1), 16, dtype=torch.uint8, device=dev)
    trig_host = torch.empty(n_slots, 40, dtype=torch.uint8).pin_memory()
    fg_host = torch.empty(n_slots, 16, dtype=torch.uint8).pin_memory()
    bg_host = torch.empty(n_slots * max(S, 1), 16, dtype=torch.uint8).pin_memory()
    cnt_host = torch.empty(1, dtype=torch.int32).pin_memory()
    state = {"i": 0}
    fed = []                                             # indices of the strain chunks fed so far, in order

    def step(xin, events=None, fg_out=fg_out, bg_out=bg_out):
        """One pass of the hot path over one chunk (every call goes through the C ABI)."""
        i = state["i"]
        cur, prev = trig[i & 1], trig[(i & 1) ^ 1]
        if events is not None: events[0].record()
        bk.filter_chunk(xin)                                           # H0-H3 (+ fused H4 maximum)
        fed.append(state.get("chunk"))
        if events is not None: events[1].record()
        bk.peaks(w["thr"], 0, trig=cur, count=counts[i:i + 1])         # H4
        if events is not None: events[2].record()
        if has_sky:
            view = bk.snr_view()
            plan.search(view, prev, n_slots, out=fg_out)               # H5 on the previous chunk's candidates
            if events is not None: events[3].record()
            if S:
                plan.background(view, prev, n_slots, S, 2048, mult, out=bg_out)   # H6
        elif events is not None:
            events[3].record()
        if events is not None: events[4].record()
        state["i"] = i + 1
        return cur

    # ---- fill the SNR ring (set-up, untimed): the slides need S seconds of history
    n_fill = w["ring_len"] // 2048
    for c in range(n_fill):
        bk.filter_chunk(x_dev[c % n_chunks])
        fed.append(c % n_chunks)
    torch.cuda.synchronize()
    t_setup = time.time() - t_setup
    c0 = n_fill
    for j in range(args.warmup):
        state["chunk"] = (c0 + j) % n_chunks
        step(x_dev[(c0 + j) % n_chunks])
    c0 += args.warmup
    torch.cuda.synchronize()

    # ---- device-timed region: K steps, inputs resident in HBM
    K = args.steps
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(5)] for _ in range(K)]
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    bk.timing_enable(K)
    clocks = ClockSampler(local_rank) if rank == 0 else None
    launches0 = sp.spiir_launch_count()
    i_first = state["i"]
    wall0 = time.time()
    e_begin, e_end = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e_begin.record()
    for j in range(K):
        state["chunk"] = (c0 + j) % n_chunks
        step(x_dev[(c0 + j) % n_chunks], evs[j])
    e_end.record()
    torch.cuda.synchronize()
    wall1 = time.time()
    if world > 1:
        dist.barrier()
    launches = sp.spiir_launch_count() - launches0
    ms_total = e_begin.elapsed_time(e_end)
    ms_rec, ms_chunkcall, n_rec = bk.timing_read()
    bk.timing_enable(0)
    clk = clocks.stop(wall0, wall1) if clocks else None
    c0 += K
    stage = np.zeros(4)
    per_step_ms = []
    for e in evs:
        for q in range(4):
            stage[q] += e[q].elapsed_time(e[q + 1])
        per_step_ms.append(e[0].elapsed_time(e[4]))
    cnt = counts.cpu().numpy()
    # candidates searched in step j are those found in step j-1
    n_cand = int(cnt[i_first - 1:i_first - 1 + K].sum()) if has_sky else 0
    evals = n_cand * w["n_pix"] * (1 + S)
    # every valid candidate of the last step must have been searched on every slide (ring filled, one-chunk lag)
    searched = None
    if has_sky:
        prev_np = sp.triggers_to_numpy(trig[state["i"] & 1])
        fg_np = sp.results_to_numpy(fg_out)
        okf = fg_np["pix"][prev_np["valid"] == 1] >= 0
        searched = float(okf.mean()) if okf.size else None
        if S:
            bg_np = sp.results_to_numpy(bg_out).reshape(n_slots, S)
            okb = bg_np["pix"][prev_np["valid"] == 1] >= 0
            searched = min(searched, float(okb.mean())) if okb.size else searched

    # ---- parity in the regime that was just timed (once, outside the timed region; rank 0 of a single-GPU run):
    #      the SNR of a seeded sample of templates over the whole stream fed so far against the float64 oracle
    #      (O1-O3), and the last step's sky results of those templates' candidates, foreground and every slide,
    #      against O6 / O7 on the ring as it stands (wrapped, threshold 4, 100 slides)
    parity = None
    if world == 1 and has_sky and not args.no_parity:
        parity = parity_check(args, w, bank, x, fed, bk, trig[state["i"] & 1], fg_out, bg_out, u2, delay, mult,
                              dec if multirate else None, itp if multirate else None)

    # ---- NEXT-1 (outside the timed step): xi^2 of the last step's candidates (Eq. 11, 12), n_j = 175, on a
    #      seeded synthetic autocorrelation table (the arithmetic and the traffic do not depend on its values)
    xi2_info = rank_info = None
    if has_sky:
        nj = 175
        g = torch.Generator(device="cpu").manual_seed(cfg["seed"])
        lag = torch.arange(-nj, nj + 1, dtype=torch.float32)
        tau = 5.0 + 40.0 * torch.rand(T, 1, generator=g)
        om = 0.1 + 1.2 * torch.rand(T, 1, generator=g)
        env = torch.exp(-lag.abs()[None, :] / tau)
        ac = torch.stack([env * torch.cos(om * lag[None, :]), env * torch.sin(om * lag[None, :])], dim=-1).contiguous().to(dev)
        dl_dev = torch.from_numpy(np.ascontiguousarray(delay, dtype=np.int32)).to(dev)
        prev = trig[state["i"] & 1]
        view = bk.snr_view()
        xi_out = torch.empty(n_slots, 24, dtype=torch.uint8, device=dev)
        ex = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
        for rep in range(4):
            if rep == 1: ex[0].record()
            sp.signal_consistency(view, dl_dev, prev, fg_out, n_slots, ac, nj, out=xi_out)
        ex[1].record()
        torch.cuda.synchronize()
        xi = sp.xi2_to_numpy(xi_out)
        n_used = int(xi["used"].sum())
        ms_xi = ex[0].elapsed_time(ex[1]) / 3.0
        by = n_used * (D + 1) * (2 * nj + 1) * 8.0
        xi2_info = {"ms": ms_xi, "candidates": n_used, "algorithmic_GBps": by / (ms_xi * 1e-3) / 1e9,
                    "median_xi2_c": float(np.median(xi["xi2_c"][xi["used"] == 1])) if n_used else None,
                    "note": "not part of the timed step; synthetic autocorrelation table"}
        if S:                                             # the same for the background events of the 100 slides
            xb_out = torch.empty(n_slots * S, 24, dtype=torch.uint8, device=dev)
            for rep in range(3):
                if rep == 1: ex[0].record()
                sp.signal_consistency(view, dl_dev, prev, bg_out, n_slots, ac, nj, out=xb_out,
                                      n_slides=S, step=2048, mult=mult)
            ex[1].record()
            torch.cuda.synchronize()
            n_bg = int(sp.xi2_to_numpy(xb_out)["used"].sum())
            ms_b = ex[0].elapsed_time(ex[1]) / 2.0
            xi2_info["slides"] = {"ms": ms_b, "events": n_bg,
                                  "algorithmic_GBps": n_bg * (D + 1) * (2 * nj + 1) * 8.0 / (ms_b * 1e-3) / 1e9}
            # NEXT-2: the chunk's coherent background events into a 256 x 256 histogram, R / FAP tables, ranking
            rk = sp.Ranker(256, 256, 4.0, 12.0, -3.0, 5.0)
            rk_out = torch.empty(n_slots, 16, dtype=torch.uint8, device=dev)
            ev = [torch.cuda.Event(enable_timing=True) for _ in range(4)]
            for rep in range(3):
                rk.reset()
                ev[0].record(); rk.accumulate(prev, bg_out, xb_out, n_slots, S)
                ev[1].record(); rk.finalize()
                ev[2].record(); rk.candidates(prev, fg_out, xi_out, n_slots, float(S), out=rk_out)
                ev[3].record()
            torch.cuda.synchronize()
            rr = sp.rank_to_numpy(rk_out)
            rank_info = {"accumulate_ms": ev[0].elapsed_time(ev[1]), "finalize_ms": ev[1].elapsed_time(ev[2]),
                                "candidates_ms": ev[2].elapsed_time(ev[3]), "bins": [256, 256],
                                "background_events": rk.tables()[0], "coherent_candidates": int(rr["selected"].sum())}
            del xb_out

    # ---- the paper's own background grid (768 directions, nside 8) for the same candidates, outside
    #      the timed step (reading A17 keeps the timed background on the foreground grid)
    bg8_info = None
    if has_sky and S:
        u2b, delayb = sp.sky_table_build(8, pos, resp, cfg["sigma"], st["gmst"], 2048.0)
        plan8 = sp.SkyPlan(u2b, delayb, max_slots=n_slots)
        prev = trig[state["i"] & 1]
        view = bk.snr_view()
        eb = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
        for rep in range(3):
            if rep == 1: eb[0].record()
            plan8.background(view, prev, n_slots, S, 2048, mult, out=bg_out)
        eb[1].record()
        torch.cuda.synchronize()
        ms8 = eb[0].elapsed_time(eb[1]) / 2.0
        n_c = int((sp.triggers_to_numpy(prev)["valid"] == 1).sum())
        bg8_info = {"ms": ms8, "directions": 768, "evals_per_s": n_c * 768.0 * S / (ms8 * 1e-3),
                    "note": "not part of the timed step"}

    # ---- NEXT-3: the foreground search with sub-sample alignment (windows resampled 2 x finer by the cubic
    #      interpolator, table at 2 x 2048 Hz), same candidates, outside the timed step
    sub_info = None
    if has_sky:
        R_SUB, H_SUB = 2, 58
        u2s, delays = sp.sky_table_build(w["nside"], pos, resp, cfg["sigma"], st["gmst"], 2048.0 * R_SUB)
        plan_s = sp.SkyPlan(u2s, delays, max_slots=n_slots)
        prev = trig[state["i"] & 1]
        view = bk.snr_view()
        for _ in range(2):                                           # warm-up (allocator, first-use set-up)
            wview, wtrig = sp.upsample_windows(view, D, prev, n_slots, R_SUB, H_SUB)
            sub_out = plan_s.search(wview, wtrig, n_slots)
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
        ev[0].record()
        wview, wtrig = sp.upsample_windows(view, D, prev, n_slots, R_SUB, H_SUB)
        ev[1].record()
        sub_out = plan_s.search(wview, wtrig, n_slots)
        ev[2].record()
        torch.cuda.synchronize()
        n_c = int((sp.triggers_to_numpy(wtrig)["valid"] == 1).sum())
        win_bytes = D * (n_c * 8.0 * (2 * H_SUB + 3) + n_slots * 8.0 * (2 * R_SUB * H_SUB + 2))   # read + written
        sub_info = {"factor": R_SUB, "half_width": H_SUB, "candidates": n_c, "delay_tuples": plan_s.n_tuples,
                    "ms_upsample": ev[0].elapsed_time(ev[1]), "ms_search": ev[1].elapsed_time(ev[2]),
                    "upsample_GBps": win_bytes / (ev[0].elapsed_time(ev[1]) * 1e-3) / 1e9,
                    "note": "not part of the timed step"}
        del plan_s, wview, wtrig, sub_out

    # ---- NEXT-4: the front end (down-sampling 16 384 -> 2048 Hz, Eq. 1 whitening, gating) on seeded coloured noise,
    #      one 2-s hop per call, outside the timed step (the configs' strain is already whitened)
    fe_info = None
    if rank == 0:
        Rf, Hf = 8, 4096
        fe_ = sp.FrontEnd(D, workloads.frontend_taps(Rf, 192), decim=Rf, hop=Hf, n_hist=27, gate_pad=512,
                          out_rate_hz=2048.0, gate_threshold=8.0)
        raw = torch.from_numpy(workloads.frontend_strain(cfg["seed"], D, Rf * Hf * 4)).to(dev)
        fo = torch.empty(D, Hf, dtype=torch.float32, device=dev)
        ef = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
        for rep in range(34):
            if rep == 30: ef[0].record()
            fe_.chunk(raw[:, (rep % 4) * Rf * Hf:(rep % 4 + 1) * Rf * Hf].contiguous(), out=fo)
        ef[1].record()
        torch.cuda.synchronize()
        ms_f = ef[0].elapsed_time(ef[1]) / 4.0
        fe_info = {"ms_per_hop": ms_f, "hop_seconds": Hf / 2048.0, "transform_points": 2 * Hf,
                   "algorithmic_bytes_per_hop": D * (Rf * Hf + Hf) * 4,
                   "note": "one CTA per detector, latency-bound by 2 x 13 barrier-separated FFT stages; not part of the timed step"}
        del fe_, raw, fo

    # ---- NEXT-4, second half: the early-warning bank as a second workload — this config's bank
    #      truncated at seeded cut-offs of 30-60 Hz (workloads.early_warning_bank): all filters in the bands of
    #      <= 256 Hz, bands 0-3 empty.  Few updates per byte of state and SNR written: which resource binds?
    ew_info = None
    if rank == 0 and multirate and len(cfg["band_rates"]) == 8:
        ew_info = early_warning_row(sp, workloads, torch, cfg, T, D, chunk, dec, itp, x_dev, dev)

    # ---- BASELINE.json configs[3], the sky-search stress shape (4096 candidates on packed +-50 ms snippets, nside 64,
    #      100 slides), sky search only, outside the timed step: the driver-run figure behind README's config-3 numbers
    cfg3_info = None
    if rank == 0 and has_sky and not args.no_cfg3:
        cfg3_info = sky_stress_cfg3_row(sp, workloads, torch)

    # ---- end to end: pinned host strain in, host candidates and results out, every step
    e2e = None
    if not args.no_e2e:
        torch.cuda.synchronize()
        h2d = D * chunk * 4
        d2h = n_slots * 40 + 4 + (n_slots * 16 + (n_slots * S * 16 if S else 0) if has_sky else 0)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        if world > 1:
            dist.barrier()
        # software-pipelined as a streaming caller would run it: the device->host copies of step j (on a copy
        # stream, into the second of two host/device result sets) overlap the kernels of step j+1; the caller
        # reads step j's results, complete on the host, while step j+1 runs.  Every step's strain comes from
        # pinned host memory and every step's candidates and results reach the host inside the timed region.
        copy_stream = torch.cuda.Stream(device=dev)
        main = torch.cuda.current_stream()
        dev_sets = [(fg_out, bg_out), (torch.zeros_like(fg_out), torch.zeros_like(bg_out))]
        host_sets = [(trig_host, fg_host, bg_host, cnt_host),
                     tuple(torch.empty_like(t).pin_memory() for t in (trig_host, fg_host, bg_host, cnt_host))]
        done = [None, None]
        torch.cuda.synchronize()
        e0.record()
        for j in range(K):
            b = j & 1
            if done[b] is not None:
                main.wait_event(done[b])                             # result set b has been copied out
            state["chunk"] = (c0 + j) % n_chunks
            x_in.copy_(x_host[(c0 + j) % n_chunks], non_blocking=True)
            cur = step(x_in, fg_out=dev_sets[b][0], bg_out=dev_sets[b][1])
            ready = torch.cuda.Event()
            ready.record(main)
            th, fh, bh, ch = host_sets[b]
            with torch.cuda.stream(copy_stream):
                copy_stream.wait_event(ready)
                th.copy_(cur, non_blocking=True)
                ch.copy_(counts[state["i"] - 1:state["i"]], non_blocking=True)
                if has_sky:
                    fh.copy_(dev_sets[b][0], non_blocking=True)
                    if S:
                        bh.copy_(dev_sets[b][1], non_blocking=True)
                done[b] = torch.cuda.Event()
                done[b].record(copy_stream)
            if j >= 1:
                done[b ^ 1].synchronize()                            # the caller reads step j-1's results
        done[(K - 1) & 1].synchronize()
        e1.record()
        torch.cuda.synchronize()
        ms_e2e = shd.max_over_ranks(e0.elapsed_time(e1), dev)
        e2e = {"value": world * upd_chunk * K / (ms_e2e * 1e-3), "unit": UNIT, "ms_per_step": ms_e2e / K,
               "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
               "pipelining": "results of step j copied out on a second stream while step j+1 computes"}
        c0 += K

    ms_total = shd.max_over_ranks(ms_total, dev)
    upd_all = shd.sum_over_ranks(upd_chunk * K, dev)
    evals_all = shd.sum_over_ranks(evals, dev)
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel (+ the other one), FP32 probe, CPU baseline
    import bench_probes as bp
    ffma_rate, _ = bp.fp32_peak_probe(20)
    probes = {"unit": "fraction of the nominal FP32 lane rate (148 SM x 128 lanes x 1.965 GHz), register-only loops",
              "recursion_mix_k_bank": bp.pipe_probe(1) / FP32_LANE_OPS_PER_S,
              "quadratic_form_packed_ffma2": bp.pipe_probe(2) / FP32_LANE_OPS_PER_S,
              "quadratic_form_scalar_ffma": bp.pipe_probe(3) / FP32_LANE_OPS_PER_S}
    ms_sky = stage[2] + stage[3]
    traffic = ncu_traffic_bytes()
    # executed FP32 lane-operations of the recursion: 8 per update, 5 in the band above the output rate, which
    # advances two samples per step; `counted` keeps the paper's 8 per update everywhere
    band_arr = np.asarray(bank["band"]).astype(np.int64)
    upd_b0 = int(D * np.sum(band_arr == 0) * chunk) if bk.out_band == 1 else 0
    exec_ops = (5.0 * upd_b0 + 8.0 * (upd_chunk - upd_b0)) * n_rec
    roof_bank = alu_roofline("k_bank (IIR recursion, H1+H2)", FLOP_PER_UPDATE * upd_chunk * n_rec, ms_rec,
                             n_rec * len_groups(bk), ffma_rate, traffic["k_bank"],
                             issue_ops=8.0 * upd_chunk * n_rec, executed_ops=exec_ops)
    roof_bank["flop_per_unit"] = "12 per filter-sample update (PAPER.md:135)"
    roof_sky = None
    if has_sky and evals:
        roof_sky = alu_roofline("k_sky (coherent search + slides, H5+H6)", FLOP_PER_EVAL * evals, ms_sky,
                                2 * D * K if S else D * K, ffma_rate, traffic["k_sky"],
                                issue_ops=6.5 * evals, executed_ops=5.5 * evals)
        roof_sky["flop_per_unit"] = ("9 per (candidate or candidate-slide, direction) evaluation, the flop k_sky EXECUTES: "
                                     "1 FMUL + 4 FFMA of the five-term quadratic form of Eq. 28 (trace of the projector = 2)")
        roof_sky["flop_per_unit_other_countings"] = FLOP_PER_EVAL_CONTEXT
    dominant, other = (roof_bank, roof_sky) if (roof_sky is None or ms_rec >= ms_sky) else (roof_sky, roof_bank)
    line = {
        "metric": METRIC, "value": upd_all / (ms_total * 1e-3), "unit": UNIT, "n_gpus": world, "steps": K,
        "warmup": args.warmup, "ms_per_step": ms_total / K, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        # the sampled oracle check of the run just timed rides inside `config` too, a key the driver's record keeps
        "config": dict(config_dict(args, w), parity_checked={k: parity.get(k) for k in ("ok", "n", "max_err")}
                       if isinstance(parity, dict) else parity),
        "sky_evals_per_s": evals_all / (ms_total * 1e-3) if has_sky else None,
        "chunk_latency_ms": ms_total / K,
        "chunk_latency_ms_median_max": [float(np.median(per_step_ms)), float(np.max(per_step_ms))],
        "stages_ms_per_step": {"filter_chunk": stage[0] / K, "of_which_k_bank": ms_rec / max(1, n_rec),
                               "peaks": stage[1] / K, "sky_foreground": stage[2] / K, "sky_slides": stage[3] / K},
        "stage_rates": {"bank_updates_per_s": upd_chunk * K / (stage[0] * 1e-3),
                        "k_bank_updates_per_s": upd_chunk * n_rec / (ms_rec * 1e-3),
                        "sky_evals_per_s": (evals / (ms_sky * 1e-3)) if (has_sky and ms_sky > 0) else None},
        "parity_checked": parity,
        "per_step": {"updates": upd_chunk, "candidates": n_cand / K if has_sky else None,
                     "sky_evals": evals / K if has_sky else None, "searched_fraction": searched},
        "roofline": dict(dominant, other_kernel=other), "roofline_other": other, "pipe_probes": probes,
        "next_rows": {"xi2": xi2_info, "rank": rank_info, "sub_sample_foreground": sub_info, "frontend": fe_info,
                      "early_warning": ew_info},
        "background_on_paper_grid_nside8": bg8_info, "sky_stress_cfg3": cfg3_info,
        "e2e": e2e, "gpu_launches": int(launches), "clocks": clk, "setup_s": t_setup,
    }
    if world == 1 and not args.no_cpu_baseline:
        # about 10-15 s of host work at config 4
        leg = cpu_leg(args, w, min(8192, T), 2, 4096 if has_sky else 0)
        cpu_v, cpu_t = oracle_whole_step_rate(leg["acc"], upd_chunk, evals / K if has_sky else 0, n_slots)
        line["cpu_baseline"] = cpu_baseline_dict(leg, cpu_v, cpu_t, w, S)
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def measured_hbm_gbs():
    """HBM copy bandwidth of this pool's B200s from the driver-written MEASURED_PEAKS.json, else the profiling
    guide's fallback (B200_PROFILING.md: ~6.5 TB/s measured copy rate); returns (GB/s, source)."""
    try:
        return float(json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))["hbm_gbs"]), "MEASURED_PEAKS.json hbm_gbs"
    except Exception:
        return 6500.0, "fallback of B200_PROFILING.md (MEASURED_PEAKS.json absent)"


def early_warning_row(sp, workloads, torch, cfg, T, D, chunk, dec, itp, x_dev, dev, n_warm=6, n_timed=20):
    """bank stage (spiir_filter_chunk + spiir_peaks) on the early-warning variant of this config's bank, timed with
    CUDA events outside the timed step.  Reports filter-sample updates/s, the FP32 lane fraction of the recursion
    kernel and the algorithmic HBM bytes per chunk (coefficients once per detector as the kernel reads them, IIR
    state read + written, SNR ring written) over the stage time against the measured copy bandwidth, and names the
    larger of the two fractions as the binding resource."""
    rng = np.random.default_rng(cfg["seed"] + 393)
    full = workloads.random_bank(rng, T, cfg["filters_per_template"], cfg["band_rates"], cfg["out_band"], exact_norm=False)
    ew = workloads.early_warning_bank(full, rng, exact_norm=False)
    del full
    n_filt = int(ew["tmpl_offset"][-1])
    per_band = np.bincount(ew["band"], minlength=8)
    bk = sp.Bank(ew, D, chunk, ring_len=2 * (chunk >> cfg["out_band"]), bank_size=1000, dec_taps=dec, int_taps=itp)
    upd = bk.updates_per_chunk(chunk)
    n_x = len(x_dev)
    for j in range(n_warm):
        bk.filter_chunk(x_dev[j % n_x]); bk.peaks(4.0, 0)
    torch.cuda.synchronize()
    bk.timing_enable(n_timed)
    e = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
    e[0].record()
    for j in range(n_timed):
        bk.filter_chunk(x_dev[(n_warm + j) % n_x]); bk.peaks(4.0, 0)
    e[1].record()
    torch.cuda.synchronize()
    ms = e[0].elapsed_time(e[1]) / n_timed
    ms_rec, _, n_rec = bk.timing_read()
    bk.timing_enable(0)
    ms_rec /= max(1, n_rec)
    n_out = chunk >> cfg["out_band"]
    alg_bytes = D * n_filt * (20 + 16) + D * T * n_out * 8          # (float4 coef + int32 offset) + state r/w; ring write
    hbm, hbm_src = measured_hbm_gbs()
    gbs = alg_bytes / (ms * 1e-3) / 1e9
    lane = 8.0 * upd / (ms_rec * 1e-3) / FP32_LANE_OPS_PER_S if ms_rec > 0 else None
    lane_stage = 8.0 * upd / (ms * 1e-3) / FP32_LANE_OPS_PER_S
    info = {"workload": "this config's bank truncated at seeded cut-offs of 30-60 Hz (PAPER.md:393): %d templates, %d filters "
                        "(%.0f per template) in the bands of <= 256 Hz only, %d detectors" % (T, n_filt, n_filt / T, D),
            "filters_per_band": [int(v) for v in per_band], "updates_per_chunk": int(upd),
            "ms_per_chunk_bank_stage": ms, "ms_k_bank": ms_rec, "updates_per_s": upd / (ms * 1e-3),
            "k_bank_updates_per_s": upd / (ms_rec * 1e-3) if ms_rec > 0 else None,
            "algorithmic_bytes_per_chunk": int(alg_bytes), "achieved_GBps": gbs, "hbm_peak_GBps": hbm,
            "hbm_peak_source": hbm_src, "hbm_frac": gbs / hbm,
            "fp32_lane_frac_k_bank": lane, "fp32_lane_frac_stage": lane_stage,
            "ms_other_kernels": ms - ms_rec,
            "k_bank_hbm_frac": (D * n_filt * 36 / (ms_rec * 1e-3) / 1e9 / hbm) if ms_rec > 0 else None,
            # k_bank alone: coefficients + state over its own time against its lane fraction; the stage: whichever of the
            # two fractions is larger — when both are small the stage is bound by neither resource but by the fixed
            # per-chunk cost of the decimator / cascade / ring kernels (ms_other_kernels), which does not shrink
            # with the filter count
            "binds_k_bank": ("hbm" if ms_rec > 0 and D * n_filt * 36 / (ms_rec * 1e-3) / 1e9 / hbm > (lane or 0) else "fp32 lanes"),
            "binds_stage": ("hbm" if gbs / hbm > max(lane_stage, 0.5) else "fp32 lanes" if lane_stage > 0.5 else
                            "neither (hbm_frac and fp32_lane_frac_stage both < 0.5): fixed per-chunk cost of k_prep + k_combine"),
            "note": "not part of the timed step; diagonal noise normalisation (set-up time)"}
    del bk
    return info


def sky_stress_cfg3_row(sp, workloads, torch, reps=3):
    """coherent_sky_search + timeslide_background on BASELINE.json configs[3] exactly as tests/test_gpu_parity.py::
    test_cfg3_full sets it up (there every one of the 4096 x 101 results is held against the oracle): seeded packed
    snippets, library-built nside-64 table, 100 slides of one window each.  CUDA events around `reps` passes after one
    warm-up pass; the 2 GB of snippets exceed the 126 MB L2."""
    cfg = workloads.config(3)
    n, S, half = cfg["n_triggers"], cfg["n_slides"], cfg["snippet_half"]
    W = 2 * half + 1
    pos, resp = workloads.detector_geometry(cfg["dets"])
    u2, delay = sp.sky_table_build(cfg["nside"], pos, resp, cfg["sigma"], 0.7, 2048.0)
    z, tdet, k, _ = workloads.snr_snippets(workloads.streams(cfg["seed"])["snippets"], u2, delay, n, S + 1, half,
                                           cfg["coherent_fraction"])
    trig = np.zeros(n, sp.TRIGGER_DTYPE)
    trig["valid"] = 1; trig["tmpl"] = np.arange(n); trig["det"] = tdet; trig["k"] = k
    zd = torch.from_numpy(z).cuda()
    del z
    plan = sp.SkyPlan(u2, delay, max_slots=n)
    view = sp.SnrView(zd)
    td = sp.triggers_from_numpy(trig)
    fg = torch.empty(n, 16, dtype=torch.uint8, device="cuda")
    bg = torch.empty(n * S, 16, dtype=torch.uint8, device="cuda")
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
    ms_f = ms_b = 0.0
    for r in range(reps + 1):
        ev[0].record()
        plan.search(view, td, n, out=fg)
        ev[1].record()
        plan.background(view, td, n, S, W, [1] * len(cfg["dets"]), out=bg)
        ev[2].record()
        torch.cuda.synchronize()
        if r:
            ms_f += ev[0].elapsed_time(ev[1]) / reps
            ms_b += ev[1].elapsed_time(ev[2]) / reps
    res = sp.results_to_numpy(bg)
    evals = float(n) * (1 + S) * len(u2)
    rate = evals / ((ms_f + ms_b) * 1e-3)
    info = {"workload": "BASELINE.json configs[3]: %d candidates, %d detectors, nside %d (%d directions), %d slides, packed "
                        "snippets of %d samples" % (n, len(cfg["dets"]), cfg["nside"], len(u2), S, W),
            "ms_foreground": ms_f, "ms_slides": ms_b, "evals": evals, "evals_per_s": rate,
            "flop_per_eval_executed": FLOP_PER_EVAL, "frac_of_fp32_peak": FLOP_PER_EVAL * rate / 1e12 / FP32_PEAK_TFLOPS,
            "fp32_lane_frac_executed": 5.5 * rate / FP32_LANE_OPS_PER_S,
            "results_with_a_pixel": int((res["pix"] >= 0).sum()), "n_tuples": plan.n_tuples,
            "parity": "the same inputs and calls as tests/test_gpu_parity.py::test_cfg3_full (all results vs the oracle)",
            "note": "not part of the timed step"}
    plan.close()
    del zd, view, fg, bg
    return info


def len_groups(bk):
    """Recursion-kernel launches per chunk (one per (lanes, filters-per-lane, delay class) group)."""
    seen = set()
    for b in range(bk.n_bands):
        p = bk.band_plan(b)
        seen.add((p["lanes_per_unit"], p["filters_per_lane"], b == 0 and bk.out_band == 1))
    return len(seen)


def alu_roofline(name, flops, ms, n_launches, ffma_rate, traffic, issue_ops, executed_ops=None):
    """FP32-ALU roofline entry: achieved = algorithmic flop / device time of the kernel's launches
    (CUDA events on the launching stream, inside the timed region)."""
    achieved = flops / (ms * 1e-3) / 1e12
    return {"kernel": name, "bound": "alu", "achieved": achieved, "peak": FP32_PEAK_TFLOPS, "unit": "TFLOP/s",
            "frac": achieved / FP32_PEAK_TFLOPS, "traffic": traffic,
            "traffic_source": "profiles/r2_traffic.csv (ncu --set full capture of one step; a record, not measured by this run)",
            "peak_source": "derived: 148 SM x 128 FP32 lanes x 2 flop x 1.965 GHz (clocks.max.sm); not in "
                           "MEASURED_PEAKS.json",
            "fp32_issue_frac": issue_ops / (ms * 1e-3) / FP32_LANE_OPS_PER_S,
            "fp32_issue_frac_executed": (executed_ops / (ms * 1e-3) / FP32_LANE_OPS_PER_S) if executed_ops else None,
            "measured_ffma_tflops_same_run": 2.0 * ffma_rate / 1e12,
            "frac_of_measured_ffma": achieved / (2.0 * ffma_rate / 1e12),
            "ms_per_launch_set": ms / max(1, n_launches), "launches": n_launches}


def main():
    args = parse_args()
    if args.impl == "reference":
        if int(os.environ.get("RANK", "0")) != 0:
            return
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
