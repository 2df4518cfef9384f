#!/usr/bin/env python
"""Writes the parity report: the CUDA path (through the C ABI) against the CPU oracle per config / frame / iteration
count, with the fp32 floor (the oracle's own float instantiation against its double one) next to every number.

    python tests/parity_report.py [--out gpurun_out/parity_report.md] [--quick]

Run on a B200 box; every expected value is computed here by `oracle/` (nothing is stored, nothing comes from the CUDA
path).  The committed copy is profiles/r02_parity_report.md.  The rule that turns these numbers into pass / fail is
tests/parity_cases.py (also used by tests/test_gpu_parity.py).
"""
from __future__ import annotations

import argparse
import os
import sys
import time

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

from paper_1702_07740_b200 import workloads as W  # noqa: E402
from tests import parity_cases as PC  # noqa: E402


def fmt(x):
    return "-" if x is None else f"{x:.2e}"


def fixed_section(out, oracle, B, title, base, Z, llr, syn, iters_list, per_frame_from=PC.TOL / 10, frame_ids=None,
                  code=None):
    """One table row per iteration count + one row per frame whose floor or deviation exceeds per_frame_from."""
    out.append(f"\n### {title}\n")
    out.append("| iterations | frames | max err | median err | max fp32 floor | frames with floor > tol/2 (UNPINNED) | "
               "frames with err > tol | hard-bit mismatches where \\|L\\| > 1e-2 (pinned frames) | verdict |")
    out.append("|---|---|---|---|---|---|---|---|---|")
    detail = []
    all_ok = True
    for n_iter in iters_list:
        hard, iters, passed, post = PC.gpu_decode(B, code if code is not None else base, Z, llr, syn, n_iter, 0)
        case = PC.compare_fixed(oracle, base, Z, llr, syn, n_iter, title, hard, post, always_floor=True,
                                frame_ids=frame_ids)
        errs = np.array([f.err for f in case.frames])
        floors = np.array([f.floor for f in case.frames])
        unp = [f for f in case.frames if f.unpinned]
        over = [f for f in case.frames if f.err > PC.TOL]
        mism = sum(f.hard_mismatch for f in case.frames if not f.unpinned)
        all_ok = all_ok and case.ok
        out.append(f"| {n_iter} | {len(errs)} | {errs.max():.2e} | {np.median(errs):.2e} | {floors.max():.2e} | "
                   f"{len(unp)} | {len(over)} | {mism} | {'ok' if case.ok else 'FAIL: ' + case.failures()} |")
        for f in case.frames:
            if f.floor > per_frame_from or f.err > per_frame_from:
                detail.append(f"| {n_iter} | {f.frame} | {f.err:.2e} | {f.floor:.2e} | {f.err / max(f.floor, 1e-300):.2f} | "
                              f"{'UNPINNED' if f.unpinned else 'pinned'} | {f.hard_mismatch} of {f.decided} |")
    if detail:
        out.append(f"\nFrames whose fp32 floor or GPU deviation exceeds {per_frame_from:.0e}:\n")
        out.append("| iterations | frame | GPU err vs oracle64 | fp32 floor (oracle32 vs oracle64) | err / floor | "
                   "status | hard-bit mismatches where \\|L\\| > 1e-2 |")
        out.append("|---|---|---|---|---|---|---|")
        out.extend(detail)
    return all_ok


def stop_row(sp):
    lo, hi = PC.binomial_band_95(sp.n_frames, sp.fer_oracle)
    return (f"| {sp.label} | {sp.n_frames} | {sp.fer_gpu:.3f} | {sp.fer_oracle:.3f} | [{lo:.3f}, {hi:.3f}] | "
            f"{sp.discordant_pass} | {sp.discordant_iters} | {sp.diff_hist} | {sp.hard_mismatch_frames} | "
            f"{'yes' if sp.gpu_words_valid else 'NO'} |")


STOP_HEAD = ["| case | frames | GPU FER | oracle FER | binomial 95 % band around the oracle's | discordant pass flags | "
             "discordant iteration counts | histogram of iters_gpu - iters_oracle | decoded frames whose words differ | "
             "every GPU-passed word satisfies H x = s |", "|---|---|---|---|---|---|---|---|---|---|"]


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--out", default=os.path.join(ROOT, "gpurun_out", "parity_report.md"))
    ap.add_argument("--quick", action="store_true", help="skip the full-size sections")
    args = ap.parse_args()
    import torch
    if not torch.cuda.is_available():
        raise SystemExit("parity_report.py needs a CUDA device (there is no CPU fallback)")
    import oracle
    from paper_1702_07740_b200 import binding as B
    oracle.build()
    t0 = time.time()
    out = ["# Parity report: CUDA path vs CPU oracle (written by tests/parity_report.py on "
           f"{torch.cuda.get_device_name(0)}, {os.cpu_count()} host cores)\n",
           "Command: `python tests/parity_report.py --out gpurun_out/parity_report.md`.  err = max over variables of "
           "|L_gpu - L_oracle64| / max(1, |L_oracle64|); fp32 floor = the same for the oracle's own float instantiation "
           f"(oracle32 vs oracle64).  Tolerance {PC.TOL:g}; hard bits compared where |L_oracle64| > {PC.HARD_MIN:g}.  A frame "
           f"is UNPINNED only where its floor exceeds tol/2 = {PC.UNPINNED_AT:g}; its GPU deviation must then stay within "
           f"{PC.UNPINNED_FACTOR:g} x floor.  Everything else is held to the tolerance as stated.\n",
           "## 1. Fixed iteration count, early stop off"]
    ok = True
    cfg, base, Z, fr = W.make_config(1)
    ok &= fixed_section(out, oracle, B, "Config 1 (80x72, Z = 32, 16 frames, +1.5 dB)", base, Z, fr.llr, fr.syndrome,
                        [1, 2, 5, 10, 20, 35, 50, 80, 120])
    for ci, Zr, its in ((2, 333, [30]), (3, 1000, [30, 100, 200]), (5, 517, [40]), (3, 257, [8]), (2, 64, [12])):
        cfg, base, Z, fr = W.make_config(ci, Z=Zr, n_frames=4)
        ok &= fixed_section(out, oracle, B, f"Config {ci} structure at Z = {Zr}, 4 frames", base, Z, fr.llr,
                            fr.syndrome, its)
    if not args.quick:
        for ci in (2, 3):
            cfg, base, Z, fr = W.make_config(ci)
            ok &= fixed_section(out, oracle, B, f"Config {ci} at full size (n = 1e6, 1 frame)", base, Z, fr.llr,
                                fr.syndrome, [10, 50, 100])
        cfg, base, Z, fr = W.make_config(4, n_frames=64)
        code = B.QCLDPCCode(base, Z)
        sample = np.array([0, 9, 18, 27, 37, 45, 54, 63])
        for n_iter in (12, 50):
            hard, iters, passed, post = PC.gpu_decode(B, code, Z, fr.llr, fr.syndrome, n_iter, 0)
            case = PC.compare_fixed(oracle, base, Z, fr.llr[sample], fr.syndrome[sample], n_iter, "cfg4", hard[sample],
                                    post[sample], always_floor=True, frame_ids=sample)
            if n_iter == 12:
                out.append("\n### Config 4 (64 frames in one batch, the benched launch shape), 8 sampled frames\n")
                out.append("| iterations | frame | GPU err vs oracle64 | fp32 floor | status | hard-bit mismatches where \\|L\\| > 1e-2 |")
                out.append("|---|---|---|---|---|---|")
            for f in case.frames:
                out.append(f"| {n_iter} | {f.frame} | {f.err:.2e} | {f.floor:.2e} | "
                           f"{'UNPINNED' if f.unpinned else 'pinned'} | {f.hard_mismatch} of {f.decided} |")
            ok &= case.ok
        del code
        cfg, base, Z, fr = W.make_config(5, snr_point=3, n_frames=4)
        ok &= fixed_section(out, oracle, B, "Config 5 at full size, point 3 (+0.7 dB, mid-waterfall), 4 frames", base,
                            Z, fr.llr, fr.syndrome, [20, 50])

    out.append("\n## 2. Early stop on: pass flags, iteration counts, frame error rate\n")
    out.extend(STOP_HEAD)
    cfg, base, Z, fr = W.make_config(1)
    hard, iters, passed, _ = PC.gpu_decode(B, base, Z, fr.llr, fr.syndrome, cfg.max_iter, 1, want_posterior=False)
    sp = PC.compare_stop(oracle, base, Z, fr.llr, fr.syndrome, cfg.max_iter, "config 1, max 50", hard, iters, passed)
    out.append(stop_row(sp)); ok &= sp.discordant_pass == 0 and sp.gpu_words_valid
    for pt in range(6):
        cfg, base, Z, fr = W.make_config(5, snr_point=pt, Z=2000)
        hard, iters, passed, _ = PC.gpu_decode(B, base, Z, fr.llr, fr.syndrome, cfg.max_iter, 1, want_posterior=False)
        sp = PC.compare_stop(oracle, base, Z, fr.llr, fr.syndrome, cfg.max_iter,
                             f"config 5 structure at Z = 2000, point {pt} (+{cfg.gaps_db[pt]} dB), max 300", hard, iters,
                             passed)
        out.append(stop_row(sp)); ok &= sp.discordant_pass <= 1 and sp.gpu_words_valid
    if not args.quick:
        sample = np.array([0, 11, 21, 31])
        for pt in (3, 4, 5):
            cfg, base, Z, fr = W.make_config(5, snr_point=pt)
            hard, iters, passed, _ = PC.gpu_decode(B, base, Z, fr.llr, fr.syndrome, cfg.max_iter, 1, want_posterior=False)
            sp = PC.compare_stop(oracle, base, Z, fr.llr[sample], fr.syndrome[sample], cfg.max_iter,
                                 f"config 5 at full size, point {pt} (+{cfg.gaps_db[pt]} dB), frames {sample.tolist()} "
                                 f"of the batch of 32 (GPU batch: {int(passed.sum())}/32 pass, iterations "
                                 f"{int(iters.min())}..{int(iters.max())})", hard[sample], iters[sample], passed[sample])
            out.append(stop_row(sp)); ok &= sp.discordant_pass == 0 and sp.gpu_words_valid
    out.append(f"\nOverall: {'every case inside its bound' if ok else 'SOME CASE FAILED'}.  Wall time {time.time() - t0:.0f} s.")
    os.makedirs(os.path.dirname(args.out), exist_ok=True)
    with open(args.out, "w") as fh:
        fh.write("\n".join(out) + "\n")
    print("\n".join(out))
    return 0 if ok else 1


if __name__ == "__main__":
    sys.exit(main())
