"""Algorithmic work model of the hot path.  Pure counting, no kernels.

Per cell and per vector, n = n_p = n_q = p+1, the method of BASELINE.json's north_star
(sum factorisation with even-odd decomposed 1D contractions) executes
  * 12 contractions, each n^2 lines; one even-odd line costs ceil(n/2)^2 + floor(n/2)^2 FMA and
    4*floor(n/2) adds;
  * the quadrature-point scaling: symmetric 3x3 metric + mass factor = 3 MUL + 6 FMA + 1 MUL per point
    (general geometry), or 3 MUL + 1 MUL per point when the metric is diagonal (Cartesian cells).
An "FP64 instruction" (issue slot) is one DFMA / DADD / DMUL per lane; the B200 FP64 pipe retires
peak_tflops/2 of them per second.  Bytes: read X once + write Y once = 16 B per DoF*vector, plus
56 B per quadrature point per block of `bv` vectors for per-q-point geometry; a Chebyshev step
reads X, Y and writes X_new = 24 B per DoF*vector.
"""
from __future__ import annotations

FP64_PEAK_FALLBACK_TFLOPS = 37.1   # this repo's fe_probe_peaks on a B200 at 1965 MHz (profiles/r1_box_peaks.md)
HBM_FALLBACK_GBS = 6650.0          # B200_PROFILING.md fallback


def fp64_instr_per_cell_vec(p: int, diagonal_metric: bool, even_odd: bool = True):
    """(fma, add_or_mul) FP64 instructions per cell per vector."""
    n = p + 1
    if even_odd:
        hi, lo = (n + 1) // 2, n // 2
        fma_line, add_line = hi * hi + lo * lo, 4 * lo
    else:
        fma_line, add_line = n * n, 0
    fma = 12 * n * n * fma_line
    other = 12 * n * n * add_line
    if diagonal_metric:
        other += 4 * n ** 3
    else:
        fma += 6 * n ** 3
        other += 4 * n ** 3
    return fma, other


def work_per_dof_vec(p: int, diagonal_metric: bool, even_odd: bool = True):
    """FP64 instructions (issue slots) and flops (FMA = 2) per DoF*vector (cell work / p^3)."""
    fma, other = fp64_instr_per_cell_vec(p, diagonal_metric, even_odd)
    return (fma + other) / p ** 3, (2 * fma + other) / p ** 3


def work_per_dof_vec_oi(p: int, nq: int, diagonal_metric: bool = False):
    """The same count for n_q != n_p Gauss points per direction: rectangular
    even-odd contractions.  A line through a table with mi inputs and mo outputs costs
    ceil(mo/2) ceil(mi/2) + floor(mo/2) floor(mi/2) FMA and 2 floor(mi/2) + 2 floor(mo/2) adds (split + combine).
    Forward: N along x on n^2 lines (n -> nq), along y on nq n lines, along z on nq^2 lines; D~ (nq x nq) on nq^2 lines
    per direction; the transposes mirror them; the quadrature-point step acts on nq^3 points.
    Returns (FP64 instructions, flops) per DoF*vector."""
    n = p + 1

    def line(mi, mo):
        fma = ((mo + 1) // 2) * ((mi + 1) // 2) + (mo // 2) * (mi // 2)
        return fma, 2 * (mi // 2) + 2 * (mo // 2)

    fma = other = 0
    for lines, mi, mo in ((n * n, n, nq), (nq * n, n, nq), (nq * nq, n, nq)):       # N forward and N^T back
        f, a = line(mi, mo)
        fma += 2 * lines * f
        other += 2 * lines * a
    f, a = line(nq, nq)                                                              # D~ and D~^T, three directions
    fma += 6 * nq * nq * f
    other += 6 * nq * nq * a
    if diagonal_metric:
        other += 4 * nq ** 3
    else:
        fma += 6 * nq ** 3
        other += 4 * nq ** 3
    return (fma + other) / p ** 3, (2 * fma + other) / p ** 3


def executed_instr_per_dof_vec_cartesian(p: int) -> float:
    """FP64 instructions the Cartesian plane / line kernels actually execute per DoF*vector:
    even/odd operators chained without combine+split, Ds^T g Ds applied as the one precomputed 1D operator
    g * (Ds^T Ds).  Per line of n points: split 2h, combine 2h, mult = h(h+odd) + h^2 + odd(1+h)."""
    n = p + 1
    h, odd = n // 2, n % 2
    split = comb = 2 * h
    mult = h * (h + odd) + h * h + odd * (1 + h)
    full = split + mult + comb                                  # one complete even-odd contraction
    pass_z = split + mult + comb + mult + 6 * h + 2 * odd       # N_z, T, R = gm T + g S T
    kterm = split + mult + 4 * h + odd                          # R += g S T
    cols = split + mult + split + (2 * h + odd) + mult + comb   # R += g S T accumulated in the even/odd basis, N^T
    per_line = 2 * full + pass_z + kterm + cols + 2 * full
    return per_line * n * n / p ** 3


def bytes_per_dof_vec(p: int, per_qpoint_geometry: bool, bv: int, chebyshev: bool = False) -> float:
    n = p + 1
    b = 24.0 if chebyshev else 16.0
    if per_qpoint_geometry:
        b += 56.0 * n ** 3 / (p ** 3 * bv)
    return b


def roofline_time_s(p, ndof, nvec, diagonal_metric, per_qpoint_geometry, bv, fp64_tflops, hbm_gbs, chebyshev=False):
    """t_roof = max(bytes / BW, FP64 instructions / (peak/2))  (north_star's definition)."""
    slots, _ = work_per_dof_vec(p, diagonal_metric)
    units = float(ndof) * nvec
    t_alu = units * slots / (fp64_tflops * 1e12 / 2.0)
    t_hbm = units * bytes_per_dof_vec(p, per_qpoint_geometry, bv, chebyshev) / (hbm_gbs * 1e9)
    return max(t_alu, t_hbm), t_alu, t_hbm
