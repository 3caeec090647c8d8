"""Study for SURVEY.md 8(f).3 — FP64 H_eff.psi emulated on the low-precision tensor pipes ("AI
accelerators").  NOT on the product path: nothing in the library calls this file; it produces the error / speed table
of DESIGN.md §11 and profiles/r02_f3_emulation_study.md.

Scheme studied (Ozaki-style split-integer GEMM, the form that fits tcgen05 `kind::i8` with int32 accumulators in
TMEM): every row of the left operand and every column of the right operand gets one power-of-two scale, the scaled
entries are cut into `s` signed slices of `b` bits, A ~ sum_i 2^(-b i) A_i, and
    A B = sum_{i + j < s} 2^(-b (i + j)) A_i B_j ,
where every A_i B_j is an EXACT int8 x int8 -> int32 product; the s (s + 1) / 2 products are grouped by i + j, summed
in int32 and converted to FP64 once per group.  For H_eff.psi the contraction of an output tile runs over ALL terms of
the block (K ~ terms x sector dimension), so the row / column scales are common to the whole sum — the error is
relative to the largest term, and the mixed signs of the ~3.5 k terms (cancellation) decide how many slices the
north_star tolerance (rel-L2 <= 1e-11) needs.

Part 1 (CPU, numpy; `python -m paper_2501_18263_b200.emulation_study error`): the two GEMM phases of one H_eff.psi at
BASELINE configs[1] and a configs[2]-shaped block, operands taken from the same generators as the tests, slices held
in float64 (exact integer arithmetic), error against plain float64 as a function of s.
Part 2 (one B200; `... speed`): what the int8 tensor pipe delivers through the library GEMM (`torch._int_mm`,
cuBLASLt) on tile-shaped and large problems, the cost of slicing and recombination in plain torch ops, and the
resulting FP64-equivalent rate against cuBLAS DGEMM and the library's DMMA kernel.
"""
from __future__ import annotations

import sys
import time

import numpy as np


def split_rows(A, s, b):
    """Row-scaled b-bit slices: A ~ scale[:, None] * sum_i 2^(-b (i+1)) S_i with integer S_i, |S_i| < 2^b... the first
    slice is the integer part of A / scale * 2^b (|.| <= 2^b), the others are remainders in [-2^(b-1), 2^(b-1)]."""
    mx = np.abs(A).max(axis=1)
    e = np.where(mx > 0, np.ceil(np.log2(np.where(mx > 0, mx, 1.0))), 0.0)
    scale = 2.0 ** e
    R = A / scale[:, None]                  # |R| <= 1
    slices = []
    for i in range(s):
        R = R * 2.0 ** b
        S = np.rint(R)
        slices.append(S)
        R = R - S
    return scale, slices


def ozaki_matmul(A, B, s, b=7):
    """A @ B from s x s / 2 exact integer slice products (float64 holding small integers: sums stay below 2^53)."""
    sa, As = split_rows(A, s, b)
    sb, Bs = split_rows(B.T, s, b)
    C = np.zeros((A.shape[0], B.shape[1]))
    for g in range(s):                      # group i + j = g: one int32 accumulator in the real kernel
        acc = np.zeros_like(C)
        for i in range(g + 1):
            acc += As[i] @ Bs[g - i].T
        C += acc * 2.0 ** (-b * (g + 2))
    return C * sa[:, None] * sb[None, :]


def heff_like_problem(cfg, seed, nterms=None):
    """One output block of a two-phase H_eff.psi with realistic magnitudes: operator blocks = products of random
    isometries scaled by integral-like coefficients (mixed sign, exponential spread), psi block N(0,1)/sqrt(n)."""
    rng = np.random.default_rng(seed)
    m1, m, n, n1, T = cfg
    psi = rng.normal(size=(m, n)) / np.sqrt(m * n)
    OL = rng.normal(size=(T, m1, m)) / np.sqrt(m)
    OR = rng.normal(size=(T, n1, n)) / np.sqrt(n)
    # coefficients like V_ijkl = sum_P L^P_ij L^P_kl with |i - j| decay: log-uniform over ~4 decades, random sign
    c = 10.0 ** rng.uniform(-4.5, -0.5, size=T) * rng.choice([-1.0, 1.0], size=T)
    return psi, OL, OR, c


def run_error_study():
    print("| problem (m' x m x n x n', terms) | slices s (7 bits) | int8 products | rel-L2 phase 1 (Z) | rel-L2 of psi' block | cancellation |")
    print("|---|---|---|---|---|---|")
    for name, cfg in (("configs[1]-like 24 x 24 x 24 x 24, 900 terms", (24, 24, 24, 24, 900)),
                      ("configs[2]-like 80 x 72 x 64 x 80, 1600 terms", (80, 72, 64, 80, 1600)),
                      ("configs[3]-like 128 x 128 x 128 x 128, 3500 terms", (128, 128, 128, 128, 3500))):
        psi, OL, OR, c = heff_like_problem(cfg, 7)
        T, m1, m = OL.shape
        n1, n = OR.shape[1:]
        # exact two-phase result
        Z = OL.reshape(T * m1, m) @ psi                       # phase 1: stacked GEMM
        Zc = (c[:, None, None] * Z.reshape(T, m1, n))
        A2 = Zc.transpose(1, 0, 2).reshape(m1, T * n)          # phase 2: one GEMM over all terms
        B2 = OR.transpose(0, 2, 1).reshape(T * n, n1)
        ref = A2 @ B2
        absum = np.abs(A2) @ np.abs(B2)
        canc = np.linalg.norm(absum) / np.linalg.norm(ref)
        for s in (4, 5, 6, 7, 8):
            Ze = ozaki_matmul(OL.reshape(T * m1, m), psi, s)
            e1 = np.linalg.norm(Ze - Z) / np.linalg.norm(Z)
            Zce = (c[:, None, None] * Ze.reshape(T, m1, n)).transpose(1, 0, 2).reshape(m1, T * n)
            got = ozaki_matmul(Zce, B2, s)
            e2 = np.linalg.norm(got - ref) / np.linalg.norm(ref)
            print("| %s | %d | %d | %.1e | %.1e | %.0f |" % (name, s, s * (s + 1) // 2, e1, e2, canc))


def run_speed_study():
    import torch
    dev = torch.device("cuda", 0)

    def timed(fn, reps=10):
        for _ in range(3):
            fn()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(reps):
            fn()
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / reps * 1e-3

    print("| GEMM (M x K x N) | int8 `torch._int_mm` TOP/s | FP64 `torch.matmul` (cuBLAS DGEMM) TFLOP/s |")
    print("|---|---|---|")
    rates = {}
    for (M, K, N) in ((8192, 8192, 8192), (16384, 4096, 256), (16384, 4096, 128), (4096, 16384, 128), (2048, 2048, 2048)):
        a8 = torch.randint(-100, 100, (M, K), dtype=torch.int8, device=dev)
        b8 = torch.randint(-100, 100, (K, N), dtype=torch.int8, device=dev)
        t8 = timed(lambda: torch._int_mm(a8, b8))
        a = torch.randn(M, K, dtype=torch.float64, device=dev)
        b = torch.randn(K, N, dtype=torch.float64, device=dev)
        t64 = timed(lambda: torch.matmul(a, b), reps=3)
        rates[(M, K, N)] = (2.0 * M * K * N / t8 * 1e-12, 2.0 * M * K * N / t64 * 1e-12)
        print("| %d x %d x %d | %.0f | %.1f |" % (M, K, N, rates[(M, K, N)][0], rates[(M, K, N)][1]))

    # the whole emulated DGEMM with library pieces: slicing + s(s+1)/2 int8 GEMMs + recombination
    def split_rows_t(A, s, b=7):
        mx = A.abs().amax(dim=1)
        e = torch.where(mx > 0, torch.ceil(torch.log2(torch.where(mx > 0, mx, torch.ones_like(mx)))), torch.zeros_like(mx))
        scale = torch.pow(2.0, e)
        R = A / scale[:, None]
        out = []
        for _ in range(s):
            R = R * 2.0 ** b
            S = torch.round(R)
            out.append(S.clamp_(-127, 127).to(torch.int8))       # (|first slice| = 128 happens only for exact powers of two)
            R = R - S
        return scale, out

    def ozaki_t(A, B, s, b=7):
        sa, As = split_rows_t(A, s, b)
        sb, Bs = split_rows_t(B.t().contiguous(), s, b)
        Bs = [x.t().contiguous() for x in Bs]
        C = torch.zeros(A.shape[0], B.shape[1], dtype=torch.float64, device=A.device)
        for g in range(s):
            acc = torch._int_mm(As[0], Bs[g])
            for i in range(1, g + 1):
                acc += torch._int_mm(As[i], Bs[g - i])
            C += acc.to(torch.float64) * 2.0 ** (-b * (g + 2))
        return C * sa[:, None] * sb[None, :]

    print()
    print("| emulated DGEMM, library pieces (M = K = N = 4096) | slices | time ms | FP64-equivalent TFLOP/s | rel-L2 vs cuBLAS DGEMM |")
    print("|---|---|---|---|---|")
    M = K = N = 4096
    A = torch.randn(M, K, dtype=torch.float64, device=dev)
    B = torch.randn(K, N, dtype=torch.float64, device=dev)
    ref = A @ B
    t64 = timed(lambda: A @ B, reps=3)
    print("| cuBLAS DGEMM | - | %.2f | %.1f | - |" % (t64 * 1e3, 2.0 * M * K * N / t64 * 1e-12))
    for s in (5, 6, 7, 8):
        got = ozaki_t(A, B, s)
        err = float(torch.linalg.norm(got - ref) / torch.linalg.norm(ref))
        t = timed(lambda: ozaki_t(A, B, s), reps=3)
        tg = timed(lambda: [torch._int_mm(torch.zeros(1, device=dev).to(torch.int8).expand(M, K).contiguous(), torch.zeros(1, device=dev).to(torch.int8).expand(K, N).contiguous())], reps=1) if False else None
        print("| split-integer, int8 products only would be %.2f ms | %d | %.2f | %.1f | %.1e |" % (
            s * (s + 1) / 2 * 2.0 * M * K * N / (rates[(8192, 8192, 8192)][0] * 1e12) * 1e3, s, t * 1e3, 2.0 * M * K * N / t * 1e-12, err))


if __name__ == "__main__":
    what = sys.argv[1] if len(sys.argv) > 1 else "error"
    t0 = time.time()
    if what == "error":
        run_error_study()
    else:
        run_speed_study()
    print("\n(%.0f s)" % (time.time() - t0))
