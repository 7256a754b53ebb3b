/*
 * devmath.cuh -- device arithmetic of the hot path: oscillation terms, sin^2 of the phase,
 * energy-scale map, bin search.  Compiled with -fmad=false: every fused multiply-add below is
 * written as fma() on purpose, nothing else is contracted (bit-exact bin assignment, R8).
 */
#ifndef PHYLINO_DEVMATH_CUH
#define PHYLINO_DEVMATH_CUH

#include "internal.h"

/* -DPHYLINO_CHECKED (python -m paper_2502_15253_b200.build --checked -> libphylino_checked.so): device-side bounds
 * and invariant checks that trap with a message; compiled out of the shipped library.  compute-sanitizer is not
 * available on the measurement pool, so these stand in for memcheck on the indices the kernels compute themselves. */
#ifdef PHYLINO_CHECKED
#include <cstdio>
#define PHYLINO_ASSERT(cond)                                                                          \
    do {                                                                                              \
        if (!(cond)) {                                                                                \
            printf("PHYLINO_CHECKED %s:%d: %s (block %d thread %d)\n", __FILE__, __LINE__, #cond,     \
                   (int)blockIdx.x, (int)threadIdx.x);                                                \
            __trap();                                                                                 \
        }                                                                                             \
    } while (0)
#else
#define PHYLINO_ASSERT(cond) do { } while (0)
#endif

namespace phylino {

/* first-octant branch theta < pi/4 (R4): cos 2theta = +sqrt(1 - sin^2 2theta) */
__device__ __forceinline__ void mixing(double s22, double &cos2, double &sin2, double &cos4)
{
    double c2t = sqrt(1.0 - s22);
    cos2 = (1.0 + c2t) / 2.0;
    sin2 = (1.0 - c2t) / 2.0;
    cos4 = cos2 * cos2;
}

__device__ __forceinline__ double osc_par(const OscDev &o, const double *theta, int slot)
{
    int idx = o.idx_osc[slot];
    return idx >= 0 ? theta[idx] : o.fixed_osc[slot];
}

/* Amplitudes A_k and mass splittings dm2_k [eV^2] of the S oscillation terms at one point.
 *   EQ1      PAPER.md:34 Eq. 1
 *   FULL3    exact 3-flavour vacuum P_ee; |dm2_31|, |dm2_32| from inverting PAPER.md:39 Eq. 2 (R2, R5)
 *   STERILE4 BASELINE.json config 5 (PAPER.md:199 prints none; R15) */
__device__ __forceinline__ void osc_terms(const OscDev &o, const double *theta, double A[MAX_TERMS],
                                          double dm2[MAX_TERMS])
{
    double s13 = osc_par(o, theta, PHYLINO_S13), mee = osc_par(o, theta, PHYLINO_MEE);
    double s12 = osc_par(o, theta, PHYLINO_S12), m21 = osc_par(o, theta, PHYLINO_M21);
    double c2_13, s2_13, c4_13, c2_12, s2_12, c4_12;
    mixing(s13, c2_13, s2_13, c4_13);
    mixing(s12, c2_12, s2_12, c4_12);
    if (o.osc_model == PHYLINO_OSC_EQ1) {
        A[0] = s13;          dm2[0] = mee;
        A[1] = c4_13 * s12;  dm2[1] = m21;
        A[2] = 0.0;          dm2[2] = 0.0;
    } else if (o.osc_model == PHYLINO_OSC_FULL3) {
        /* (31, 32, 21): the slowest splitting last, as in the other models (see half_cos_small) */
        double sgn = o.ordering >= 0 ? 1.0 : -1.0;
        A[0] = s13 * c2_12;  dm2[0] = mee + sgn * s2_12 * m21;
        A[1] = s13 * s2_12;  dm2[1] = mee - sgn * c2_12 * m21;
        A[2] = c4_13 * s12;  dm2[2] = m21;
    } else {
        double s14 = osc_par(o, theta, PHYLINO_S14), m41 = osc_par(o, theta, PHYLINO_M41);
        double c2_14, s2_14, c4_14;
        mixing(s14, c2_14, s2_14, c4_14);
        A[0] = c4_14 * s13;  dm2[0] = mee;
        A[1] = s14;          dm2[1] = m41;
        A[2] = c4_13 * s12;  dm2[2] = m21;
    }
}

/* Phase in half-turns per unit x = L/E:  phase = 1.267 dm2 x  (R1)  =  (pi/2) (h x),
 * h = 1.267 dm2 (2/pi). */
__device__ __forceinline__ double halfturn_coeff(double dm2)
{
    return (1.267 * dm2) * 0.63661977236758134308;   /* 2/pi */
}

/* g(h, x) = 1/2 cos(pi h x) = 1/2 - sin^2((pi/2) h x), |h x| < 2^51, so that
 *   P_ee = 1 - sum_k A_k sin^2(phase_k) = (1 - 1/2 sum_k A_k) + sum_k A_k g(h_k, x).
 *   n = rint(h x) by the 1.5*2^52 trick, f = h x - n in [-1/2, 1/2] with ONE rounding (fma), so the
 *   range reduction is exact for phases of thousands of radians (config 5: 7.8e3 rad);
 *   1/2 cos(pi f) = 1/2 - z Q(z), z = f^2: degree-5 minimax Q, |error| <= 4.1e-13 absolute
 *   (Remez fit made for this file, checked against mpmath);
 *   cos(pi (n + f)) = (-1)^n cos(pi f): the parity of n is bit 0 of the low word of t, moved onto
 *   the sign bit of the result by ONE integer multiply-add on the high word.
 * 10 fp64 instructions + 1 integer instruction. */
__device__ __forceinline__ double half_cos_halfturns(double h, double x)
{
    const double MAGIC = 6755399441055744.0;        /* 1.5 * 2^52 */
    double t = fma(h, x, MAGIC);
    double n = t - MAGIC;
    double f = fma(h, x, -n);
    double z = f * f;
    double q =  0x1.e2a4cab0973aep-11;               /* -Q(z), Horner */
    q = fma(q, z, -0x1.a65598e5b8576p-7);
    q = fma(q, z,  0x1.e1f273f3e9df0p-4);
    q = fma(q, z, -0x1.55d3c0fdef250p-1);
    q = fma(q, z,  0x1.03c1f070b1413p+1);
    q = fma(q, z, -0x1.3bd3cc9bac6fep+1);
    double c = fma(q, z, 0.5);
    unsigned hi = (unsigned)__double2hiint(c) + ((unsigned)__double2loint(t) << 31);
    return __hiloint2double((int)hi, __double2loint(c));
}

/* The same g where the phase never leaves the first eighth of a half-turn: |h x| <= SMALL_PHASE for every event
 * of the dataset and every point of the group (decided once per call and group from max |h| and the dataset's
 * max L/E, spectra.cu).  No range reduction (n = 0, f = h x with the one rounding the general path has too) and a
 * cubic in z instead of a quintic: degree-3 minimax of (1/2 - 1/2 cos(pi sqrt z)) / z on [0, 1/64], |error| <=
 * 2.7e-14 (Remez fit made for this file, checked against mpmath at 60 digits).  That is the solar term
 * (dm2_21 = 7.5e-5 eV^2) at Double-Chooz baselines: phase <= 0.06 rad.  6 fp64 instructions instead of 10, no
 * integer one.  The models list their terms with dm2_21 last, so "the last term is slow" is the one case built. */
constexpr double SMALL_PHASE = 0.125;
__device__ __forceinline__ double half_cos_small(double h, double x)
{
    const double f = h * x;
    const double z = f * f;
    double q =  0x1.dff2bf9124181p-4;
    q = fma(q, z, -0x1.55d2effd81fecp-1);
    q = fma(q, z,  0x1.03c1f03a3f1d1p+1);
    q = fma(q, z, -0x1.3bd3cc9bc6f40p+1);
    return fma(q, z, 0.5);
}

/* g of term k of S: the cheap form for the last term when the group's flag says so */
template <int S, bool SM> __device__ __forceinline__ double half_cos_term(int k, double h, double x)
{
    return (SM && k == S - 1) ? half_cos_small(h, x) : half_cos_halfturns(h, x);
}

/* The same two functions in ACCUMULATING form, for datasets whose MC weights are all exactly 1 (every BASELINE.json
 * config).  g = (-1)^n (1/2 + q z) with q = -Q(z) the polynomial above, so over a run of N events
 *     sum_e g_e = 1/2 (N - 2 N_odd) + sum_e q_e ((-1)^n_e z_e):
 * the oscillating part goes into the run sum with the LAST Horner step itself, C' = fma(q, +-z, C') -- the sign is moved
 * onto z by the same integer multiply-add that moved it onto the result before -- and the constant part is a count: the
 * parity bit of n is shifted into a 32-bit register (one funnel shift per event), counted with one popc per straight-line
 * stretch of at most 32 events, and the flush adds 1/2 N - N_odd to C' (exact: halves of whole numbers).  One fp64
 * instruction less per event x point x term than "form g, add it" (10 instead of 11; 6 instead of 7 for the small-phase
 * form, which has no sign) for one more integer instruction, and C' = -sum sin^2(phase) + N_odd carries one rounding
 * per event of a smaller number. */
__device__ __forceinline__ void half_cos_accumulate(double h, double x, double &C, unsigned &parity)
{
    const double MAGIC = 6755399441055744.0;        /* 1.5 * 2^52 */
    double t = fma(h, x, MAGIC);
    double n = t - MAGIC;
    double f = fma(h, x, -n);
    double z = f * f;
    double q =  0x1.e2a4cab0973aep-11;
    q = fma(q, z, -0x1.a65598e5b8576p-7);
    q = fma(q, z,  0x1.e1f273f3e9df0p-4);
    q = fma(q, z, -0x1.55d3c0fdef250p-1);
    q = fma(q, z,  0x1.03c1f070b1413p+1);
    q = fma(q, z, -0x1.3bd3cc9bac6fep+1);
    const unsigned lo = (unsigned)__double2loint(t);                /* n mod 2^32 */
    const double zs = __hiloint2double((int)((unsigned)__double2hiint(z) + (lo << 31)), __double2loint(z));  /* z >= 0 */
    C = fma(q, zs, C);
    parity = __funnelshift_r(parity, lo, 1);                        /* (parity >> 1) | (n & 1) << 31 */
}

__device__ __forceinline__ void half_cos_small_accumulate(double h, double x, double &C)
{
    const double f = h * x;
    const double z = f * f;
    double q =  0x1.dff2bf9124181p-4;
    q = fma(q, z, -0x1.55d2effd81fecp-1);
    q = fma(q, z,  0x1.03c1f03a3f1d1p+1);
    q = fma(q, z, -0x1.3bd3cc9bc6f40p+1);
    C = fma(q, z, C);
}

/* ... and where |h x| <= MEDIUM_PHASE = 1/2 for every event a lane meets in a work item: n = 0, f = h x exactly as the
 * general form computes it (fma(h, x, -0) is the rounded product), so the range reduction and the sign drop out and
 * the result is BIT-IDENTICAL to the general form: 8 fp64 instructions, no integer one.  That is the first term
 * (dm2_ee) at a near detector (1.267 x 2.5e-3 x 469 m / 1.9 MeV = 0.78 rad = 0.5 half-turns) and above 4 - 4.5 MeV at
 * the far one; decided per work item and group from the load-time envelope of L/E (HintEntry::x_env). */
constexpr double MEDIUM_PHASE = 0.5;
__device__ __forceinline__ void half_cos_medium_accumulate(double h, double x, double &C)
{
    const double f = h * x;
    const double z = f * f;
    double q =  0x1.e2a4cab0973aep-11;
    q = fma(q, z, -0x1.a65598e5b8576p-7);
    q = fma(q, z,  0x1.e1f273f3e9df0p-4);
    q = fma(q, z, -0x1.55d3c0fdef250p-1);
    q = fma(q, z,  0x1.03c1f070b1413p+1);
    q = fma(q, z, -0x1.3bd3cc9bac6fep+1);
    C = fma(q, z, C);
}

/* term k of S in accumulating form: SM: the last term is small; MED: the first term never wraps */
template <int S, bool SM, bool MED>
__device__ __forceinline__ void half_cos_term_accumulate(int k, double h, double x, double &C, unsigned &parity)
{
    if (SM && k == S - 1) half_cos_small_accumulate(h, x, C);
    else if (MED && k == 0) half_cos_medium_accumulate(h, x, C);
    else                  half_cos_accumulate(h, x, C, parity);
}

/* E' = fma(fma(a2, v, a1), v, a0): the normative rounding sequence of the energy-scale map (R8). */
__device__ __forceinline__ double escale(double a0, double a1, double a2, double v)
{
    return fma(fma(a2, v, a1), v, a0);
}

/* Half-open bins [edges[b], edges[b+1]): largest b with edges[b] <= e; -1 outside or NaN (R7). */
__device__ __forceinline__ int bin_search(const double *edges, int n_bins, double e)
{
    if (!(e >= edges[0]) || !(e < edges[n_bins])) return -1;
    int lo = 0, hi = n_bins;
    while (hi - lo > 1) {
        int mid = (lo + hi) >> 1;
        if (edges[mid] <= e) lo = mid; else hi = mid;
    }
    return lo;
}

} // namespace phylino
#endif
