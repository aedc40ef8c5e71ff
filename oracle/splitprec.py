"""Split-precision complex GEMM -- CPU oracle, TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline leg may import this module; it shares no code
with paper_2606_04771_b200/.

What it states.  PAPER.md:264-270 (S2.3) reduces the arithmetic of the contractions from float64 to float32
and PAPER.md:284-286 (S2.5) accepts the result when abs delta <n_46,up> < 1e-3.  On a B200 the single-precision
matrix engine is the TF32 tensor core (1 sign, 8 exponent, 10 explicit mantissa bits), so the single-precision
variant of the contraction is the standard "3 x TF32" split (reading A-18):

    x  =  hi + lo + r,     hi = round11(x),   lo = round11(x - hi),   |r| <= 2^-22 |x|
    (round11: to 11 significant bits = the TF32 mantissa, nearest, ties away from zero, taken on the float64
    value directly -- no intermediate float32 rounding; magnitudes below 2^-126 are flushed to zero)
    a b  ~  hi_a hi_b + hi_a lo_b + lo_a hi_b                    (lo_a lo_b <= 2^-22 |a b| is dropped)

applied to the real and imaginary parts of alpha * op(A) and op(B) separately, the four real products of a
complex product accumulated in single precision.  Every product of two TF32 numbers is exact in float32 (11 + 11
significant bits), so the only rounding besides the split is the float32 accumulation, whose ORDER the hardware
does not define.  The oracle therefore
  * defines the split bit by bit (round11 on the bit pattern of the double; tf32_round is the same rounding on
    float32 input -- PTX cvt.rna.tf32.f32 -- and agrees with it on every float32 number),
  * evaluates the three-term product with float64 accumulation (zgemm_split): the value any accumulation order
    approaches, and
  * states the two bounds a kernel has to meet element by element (split_bounds):
        |C_kernel - zgemm_split|  <=  K_total 2^-23 S       (float32 accumulation, worst case, S below)
        |zgemm_split - C_exact|   <=  3.1 * 2^-22 S         (the split itself)
    with S = |alpha| (|Re A| + |Im A|) (|Re B| + |Im B|) summed over k.
Functions: tf32_round, round11, split_tf32, zgemm_split, split_bounds.
"""
import numpy as np

U_TF32 = 2.0 ** -11      # unit roundoff of TF32 (10 explicit mantissa bits, round to nearest)


def tf32_round(x):
    """Round float32 (or anything convertible) to the nearest TF32 value, ties away from zero, returned as
    float32 whose 13 low mantissa bits are zero (PTX ISA, cvt.rna.tf32.f32).  Finite inputs only."""
    f = np.ascontiguousarray(x, dtype=np.float32)
    bits = f.view(np.uint32).astype(np.uint64)
    sign = bits & np.uint64(0x80000000)
    mag = bits & np.uint64(0x7FFFFFFF)
    mag = (mag + np.uint64(0x1000)) & np.uint64(0xFFFFE000)      # add half an ulp of TF32, truncate: ties go up in magnitude
    out = (sign | mag).astype(np.uint32)
    return out.view(np.float32).reshape(f.shape)


def round11(x):
    """float64 -> float64 with at most 11 significant bits: nearest, ties away from zero (add half a unit of the
    11-bit mantissa -- bit 41 of the pattern -- and clear the 42 bits below; a carry out of the mantissa moves
    into the exponent, as it must).  |result| < 2^-126 (not a normal float32) -> 0."""
    x = np.ascontiguousarray(x, dtype=np.float64)
    bits = x.view(np.uint64)
    r = ((bits + np.uint64(1 << 41)) & np.uint64(0xFFFFFC0000000000)).view(np.float64).reshape(x.shape).copy()
    r[np.abs(r) < 2.0 ** -126] = 0.0
    return r


def split_tf32(x):
    """x (float64) -> (hi, lo), both TF32-valued float32 arrays: hi = round11(x), lo = round11(x - hi), the
    difference taken in float64 (exact: hi has 11 significant bits)."""
    x = np.asarray(x, dtype=np.float64)
    hi = round11(x)
    lo = round11(x - hi)
    return hi.astype(np.float32), lo.astype(np.float32)


def _real3(ah, al, bh, bl):
    """hi hi + hi lo + lo hi of two real matrices given as TF32 pairs, float64 accumulation."""
    ah, al, bh, bl = (m.astype(np.float64) for m in (ah, al, bh, bl))
    return ah @ bh + ah @ bl + al @ bh


def zgemm_split(segments, M, N):
    """C = sum_t alpha_t * A_t (M x K_t) @ B_t (K_t x N) for complex128 matrices A_t, B_t (already op()-ed:
    transposed / conjugated as the task says) and real alpha_t, in 3 x TF32 split arithmetic: alpha is folded
    into A before the split (as the kernel folds it while it converts the A panel)."""
    C = np.zeros((M, N), dtype=np.complex128)
    for alpha, A, B in segments:
        A = alpha * np.asarray(A, dtype=np.complex128)
        B = np.asarray(B, dtype=np.complex128)
        arh, arl = split_tf32(A.real)
        aih, ail = split_tf32(A.imag)
        brh, brl = split_tf32(B.real)
        bih, bil = split_tf32(B.imag)
        re = _real3(arh, arl, brh, brl) - _real3(aih, ail, bih, bil)
        im = _real3(arh, arl, bih, bil) + _real3(aih, ail, brh, brl)
        C += re + 1j * im
    return C


def split_bounds(segments, M, N):
    """(accumulation bound, split bound) per element, as stated in the module header."""
    S = np.zeros((M, N))
    K = 0
    for alpha, A, B in segments:
        A = np.asarray(A)
        B = np.asarray(B)
        S += abs(alpha) * (np.abs(A.real) + np.abs(A.imag)) @ (np.abs(B.real) + np.abs(B.imag))
        K += A.shape[1]
    return K * 2.0 ** -23 * S, 3.1 * 2.0 ** -22 * S
