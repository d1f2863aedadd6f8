"""Temperature scans with the protocols of the workloads (reading A13): one state carried through the
scan, `equil` discarded sweeps then `sweeps` measured sweeps per temperature, M and E taken after every measured sweep.

    python -m paper_2106_11286_b200.scan c2          # prints T, <|M|>, <E>/N, chi, C per temperature

Host-side bookkeeping only: every sweep and every reduction runs in the CUDA library.
"""
import sys

import numpy as np

from . import workloads
from .binding import Context, Lattice


def make_context(cfg, device="cuda:0", seed=None):
    if cfg["kind"] == "sphere":
        lat = Lattice.fcc_sphere(cfg["R"], cfg["K"], cfg["e"], cfg["K_surf"], cfg.get("colouring", "greedy"))
    else:
        lat = Lattice(cfg["kind"], cfg["L"])
    ctx = Context(lat, cfg["J"], cfg["K"], cfg["e"], cfg["seed"] if seed is None else seed, device=device)
    if cfg["start"] == "random":
        ctx.init_random()
    else:
        ctx.init_aligned(cfg["e"])
    return ctx


def run_scan(ctx, temperatures, sweeps, equil=0):
    """Returns a dict of arrays over the temperatures: T, absM = <|M|>, E = <E>/N, chi = N (<M^2> - <|M|>^2) / T,
    C = (<E^2> - <E>^2) / (N T^2)."""
    n = ctx.n
    out = {k: [] for k in ("T", "absM", "E", "chi", "C")}
    for T in temperatures:
        if equil:
            ctx.sweep(T, equil)
        M, E = ctx.sweep_series(T, sweeps)
        m = np.linalg.norm(M, axis=1)
        out["T"].append(T)
        out["absM"].append(m.mean())
        out["E"].append(E.mean() / n)
        out["chi"].append(n * ((m * m).mean() - m.mean() ** 2) / T)
        out["C"].append((np.mean(E * E) - E.mean() ** 2) / (n * T * T))
    return {k: np.array(v) for k, v in out.items()}


def fit_order_parameter(T, m, t_lo, t_hi, Tc_fixed=None):
    """Least squares of log m = log A + beta log(1 - T/Tc) over the points with t_lo <= 1 - T/Tc <= t_hi, scanning Tc
    (the form the paper fits in its Fig. 3), or at a given Tc.  Returns (Tc, beta, A, rms of the
    log residual, points used) or None."""
    T, m = np.asarray(T, float), np.asarray(m, float)
    best = None
    # the ordered phase reaches at least to the last temperature at which m is still a good fraction of its largest value:
    # a candidate Tc below it would cut the data down to a few points that any exponent fits
    T_ordered = max(T[m >= 0.15 * m.max()])
    for Tc in ([Tc_fixed] if Tc_fixed else np.arange(T_ordered + 0.0005, max(T) * 1.1, 0.0005)):
        t = 1.0 - T / Tc
        sel = (t >= t_lo) & (t <= t_hi)
        if sel.sum() < 4:
            continue
        x, y = np.log(t[sel]), np.log(m[sel])
        beta, logA = np.polyfit(x, y, 1)
        if not 0.05 < beta < 1.0:      # a window that fell into the disordered tail, not a power law in 1 - T/Tc
            continue
        rms = float(np.sqrt(np.mean((y - (beta * x + logA)) ** 2)))
        if best is None or rms < best[3]:
            best = (float(Tc), float(beta), float(np.exp(logA)), rms, int(sel.sum()))
    return best


def window_table(T, m, t_los=(0.002, 0.005, 0.01, 0.02, 0.05), t_his=(0.02, 0.03, 0.05, 0.1, 0.2), Tc_fixed=None):
    """The effective exponent of the fit above for a sweep of windows (the paper does not state its window):
    rows (t_lo, t_hi, Tc, beta, rms, points)."""
    rows = []
    for lo in t_los:
        for hi in t_his:
            if hi < 2.5 * lo:
                continue
            f = fit_order_parameter(T, m, lo, hi, Tc_fixed)
            if f:
                rows.append((lo, hi, f[0], f[1], f[3], f[4]))
    return rows


def print_windows(T, m, Tc_values=()):
    print("# effective exponent beta of M = A (1 - T/Tc)^beta against the fit window t_lo <= 1 - T/Tc <= t_hi")
    for Tc in (None,) + tuple(Tc_values):
        print("# Tc %s:  t_lo  t_hi  Tc  beta  rms(log)  points" % ("fitted" if Tc is None else "fixed at %.4f" % Tc))
        for r in window_table(T, m, Tc_fixed=Tc):
            print("#   %.3f  %.3f  %.4f  %.4f  %.1e  %d" % r)


def load_table(path):
    """A table written by `--sc ... --out path`: columns T, <|M|>, <E>/N, chi, C."""
    a = np.loadtxt(path, comments="#", ndmin=2)
    return {k: a[:, i] for i, k in enumerate(("T", "absM", "E", "chi", "C"))}


def throughput_vs_size(sizes, T=1.30, K=0.01, seconds=0.5):
    """The paper's Fig. 2 [PAPER.md lines 44-50]: time per attempted spin update against the system size, simple cubic,
    J = 1, K = 0.01 [P:40], at T = 0.9 T_C [P:42], random start.  Each size runs sweeps for about `seconds` after as many
    warm-up sweeps, timed with CUDA events around one hb_sweep call.  Returns rows (L, N, sweeps, Gupd/s, ns per update)."""
    import torch
    rows = []
    for L in sizes:
        ctx = make_context(dict(kind="sc", L=L, J=1.0, K=K, e=(0.0, 0.0, 1.0), seed=1, start="random"))
        n = ctx.n
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ctx.sweep(T, 8)
        a.record(); ctx.sweep(T, 8); b.record(); torch.cuda.synchronize()
        sweeps = max(8, int(seconds / (a.elapsed_time(b) * 1e-3 / 8)))
        ctx.sweep(T, sweeps)
        a.record(); ctx.sweep(T, sweeps); b.record(); torch.cuda.synchronize()
        dt = a.elapsed_time(b) * 1e-3
        rows.append((L, n, sweeps, n * sweeps / dt / 1e9, dt / (n * sweeps) * 1e9))
        ctx.close()
        del ctx
        torch.cuda.empty_cache()
    return rows


def main(argv):
    """python -m paper_2106_11286_b200.scan c2 | --sc L [--K k] [--T a:b:n] [--equil e] [--sweeps s] [--fit t_lo:t_hi]
    [--out file] [--windows [--Tc 1.443,1.445]] | --analyse file [Tc ...] | --fig2 [L ...] | --paper-scheme [L ...]"""
    if len(argv) > 1 and argv[1] == "--fig2":
        sizes = [int(x) for x in argv[2:]] or [16, 32, 64, 128, 256, 464, 512, 1024]
        print("# sc L^3, J = 1, K = 0.01, T = 1.30 (0.9 T_C), random start: attempted updates per second, time per update")
        print("# the paper (V100, its own scheme): 1.59 ns per update for N >= 2^18 [P:50], ~100 ns on a CPU [P:42]")
        print("# L  N  sweeps  Gupd/s  ns/update")
        for r in throughput_vs_size(sizes):
            print("%d  %d  %d  %.2f  %.5f" % r)
        return
    if len(argv) > 1 and argv[1] == "--paper-scheme":
        # the paper's own block scheme, emulated (hb_sweep_paper_scheme), at the parameters of its Figs. 1-2: rate against L and n
        import torch
        sizes = [int(x) for x in argv[2:]] or [128, 256, 464]
        print("# the paper's scheme (N/n blocks of n spins, one random spin per block and step [P:30-32]) emulated on this device;")
        print("# sc L^3, J = 1, K = 0.01, T = 1.30; the paper: 0.61-0.63 Gupd/s on a V100 with n = 8 [P:42-44]")
        print("# L  n  Gupd/s")
        for L in sizes:
            ctx = make_context(dict(kind="sc", L=L, J=1.0, K=0.01, e=(0.0, 0.0, 1.0), seed=1, start="random"))
            ctx.sweep(1.30, 20)
            for n in (4, 8, 16, 64):
                ctx.sweep_paper_scheme(1.30, 2, n)
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record(); ctx.sweep_paper_scheme(1.30, 10, n); b.record(); torch.cuda.synchronize()
                print("%d  %d  %.2f" % (L, n, ctx.n * 10 / (a.elapsed_time(b) * 1e-3) / 1e9))
            ctx.close()
        return
    if len(argv) > 1 and argv[1] == "--sc":
        import argparse
        ap = argparse.ArgumentParser()
        ap.add_argument("--sc", type=int, required=True)
        ap.add_argument("--K", type=float, default=0.01)
        ap.add_argument("--T", default="1.00:1.50:26")
        ap.add_argument("--equil", type=int, default=10000)
        ap.add_argument("--sweeps", type=int, default=10000)
        ap.add_argument("--fit", default="0.02:0.2")
        ap.add_argument("--out", default=None, help="also write the table (and the fits) to this file")
        ap.add_argument("--windows", action="store_true", help="the effective exponent over a sweep of fit windows")
        ap.add_argument("--Tc", default="", help="comma-separated critical temperatures to hold fixed in the window sweep")
        a = ap.parse_args(argv[1:])
        if a.out:      # everything printed below goes to the file as well
            import io
            class Tee(io.TextIOBase):
                def __init__(self, *fs): self.fs = fs
                def write(self, t):
                    for f in self.fs: f.write(t)
                    return len(t)
                def flush(self):
                    for f in self.fs: f.flush()
            sys.stdout = Tee(sys.__stdout__, open(a.out, "w"))
        lo, hi, k = a.T.split(":")
        Ts = [float(x) for x in np.linspace(float(lo), float(hi), int(k))]
        cfg = dict(kind="sc", L=a.sc, J=1.0, K=a.K, e=(0.0, 0.0, 1.0), seed=1, start="aligned")
        ctx = make_context(cfg)
        res = run_scan(ctx, Ts, a.sweeps, a.equil)
        print("# sc %d^3, K = %g, aligned start, heating, %d + %d sweeps per temperature" % (a.sc, a.K, a.equil, a.sweeps))
        print("# T  <|M|>  <E>/N  chi  C")
        for i in range(len(Ts)):
            print("%.4f  %.6f  %.6f  %.4f  %.4f" % tuple(res[k][i] for k in ("T", "absM", "E", "chi", "C")))
        t_lo, t_hi = (float(x) for x in a.fit.split(":"))
        fit = fit_order_parameter(res["T"], res["absM"], t_lo, t_hi)
        if fit:
            print("# fit M = A (1 - T/Tc)^beta over %g <= 1 - T/Tc <= %g: Tc = %.4f, beta = %.4f, A = %.4f, rms(log) = %.2e" %
                  ((t_lo, t_hi) + fit[:4]))
        if a.windows:
            print_windows(res["T"], res["absM"], [float(x) for x in a.Tc.split(",") if x])
        ctx.close()
        sys.stdout.flush()
        return
    if len(argv) > 2 and argv[1] == "--analyse":     # the fits again from a saved table (no device needed)
        res = load_table(argv[2])
        print_windows(res["T"], res["absM"], [float(x) for x in argv[3:]])
        return
    name = argv[1] if len(argv) > 1 else "c2"
    cfg = workloads.CONFIGS[name]
    ctx = make_context(cfg)
    res = run_scan(ctx, cfg["T"], cfg["sweeps"], cfg.get("equil", 0))
    print("# %s: %s, N = %d" % (name, cfg["kind"], ctx.n))
    print("# T  <|M|>  <E>/N  chi  C")
    for i in range(len(res["T"])):
        print("%.4f  %.6f  %.6f  %.4f  %.4f" % tuple(res[k][i] for k in ("T", "absM", "E", "chi", "C")))
    ctx.close()


if __name__ == "__main__":
    main(sys.argv)
