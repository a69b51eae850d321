"""Executed-flop fraction of the FP64 / FP32 peak from an ncu report (the cross-check of bench.py's roofline.frac).

    python -m paper_2106_12631_b200.ncu_fraction gpurun_out/<name>.ncu-rep [flops_per_event events_per_launch]

Reads `ncu -i <rep> --page raw --csv` (one `ncu --set full --clock-control none` capture of the sigmaKin kernel) and prints
  executed flops per launch = 2 x FMA + ADD + MUL thread instructions (DFMA/DADD/DMUL, or FFMA/FADD/FMUL for FP32 kernels),
  the cycle-normalised fraction  executed flops / (SMs x lanes x 2 x elapsed SM cycles)  (lanes: 64 FP64, 128 FP32),
  and, when the tally is given, tally x events / executed flops (must be <= 1 + a few per cent: the generator's explicit
  flop count of DESIGN.md §6 may not exceed what the hardware executed).
"""
import csv
import io
import subprocess
import sys


def read(rep):
    raw = subprocess.run(["ncu", "-i", rep, "--page", "raw", "--csv"], capture_output=True, text=True, check=True).stdout
    rows = list(csv.reader(io.StringIO(raw)))
    return [dict(zip(rows[0], r)) for r in rows[2:]], dict(zip(rows[0], rows[1]))


def fraction(d):
    cyc = float(d["sm__cycles_elapsed.max"])
    per_cycle = lambda op: float(d.get("smsp__sass_thread_inst_executed_op_%s_pred_on.sum.per_cycle_elapsed" % op, 0) or 0)
    out = {}
    for name, ops, lanes in (("fp64", ("dfma", "dadd", "dmul"), 64), ("fp32", ("ffma", "fadd", "fmul"), 128)):
        fma, add, mul = (per_cycle(o) * cyc for o in ops)
        flops = 2 * fma + add + mul
        out[name] = (flops, flops / (148 * lanes * 2 * cyc))
    return out, cyc


def main():
    rep = sys.argv[1]
    kernels, _ = read(rep)
    for d in kernels:
        f, cyc = fraction(d)
        kind = "fp64" if f["fp64"][0] >= f["fp32"][0] else "fp32"
        flops, frac = f[kind]
        line = "%s: %s, %.4e executed flops per launch, %.0f SM cycles, %.2f %% of the %s peak (cycle-normalised)" % (
            d.get("Kernel Name", "?")[:90], d.get("gpu__time_duration.sum", "?") + " " , flops, cyc, 100 * frac, kind.upper())
        if len(sys.argv) >= 4:
            tally = float(sys.argv[2]) * float(sys.argv[3])
            line += "; tally x events = %.4e = %.4f of executed" % (tally, tally / flops)
        print(line)


if __name__ == "__main__":
    main()
