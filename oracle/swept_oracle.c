/* oracle/swept_oracle.c -- CPU oracle for the swept-rule hot path.  TEST INFRASTRUCTURE ONLY.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may load
 * this library.  It shares no code with the CUDA path under paper_1612_02495_b200/ and neither
 * imports the other.
 *
 * What it computes: the plain definition of the result the swept rule must reach -- nsteps naive
 * applications of each explicit scheme on the whole periodic array, in the
 * run precision (float or double; PAPER.md:138 `REAL`), with the point-update operation order fixed
 * in DESIGN.md.  Schemes: heat FTCS (Eq. 2), Kuramoto-Sivashinsky central/RK2 (Eq. 4, 15,
 * 16 PAPER.md:64, 291, 295; sign reading G1), Euler MUSCL/minmod/Rusanov midpoint (BASELINE.json
 * config 4; not in the paper -- see DESIGN.md "Readings").
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): heat -- amplification factor 1-4r sin^2(k dx/2),
 * Pascal-triangle delta response (exact), Nyquist annihilation, sum conservation, max principle;
 * heat with insulated ends -- bitwise equal to the periodic oracle on the mirrored 2n-point rod, cosine
 * (DCT-II) modes decay by 1-4r sin^2(k pi/2n), exact dyadic hand-stepped 4-point rod, sum conservation;
 * KS -- uniform fixed point, sum conservation, linearised complex growth factor about a uniform
 * offset (pins every coefficient and sign incl. the nonlinear one), bitwise shift equivariance,
 * exact-rational nx=8 hand stepping; Euler -- conservation, uniform fixed point, mirror symmetry,
 * exact Riemann (Sod) star states, positivity, second-order convergence on an exactly advected
 * smooth density wave, TVD / no new extrema on an advected square contact (both checked to FAIL on
 * one-line mutants: zero / maxmod / unlimited slopes, full-step predictor, forward Euler, wrong face
 * sign).  Parity unpinned: none.  (Euler is BASELINE.json config 4's scheme; the paper has none.)
 *
 * 2-D heat (heat2d.inc) -- separable amplification factor 1-4Fo(sin^2+sin^2), exact lattice-walk delta response
 * at Fo = 1/4 (binomial closed form), sum conservation, max principle, bitwise transposition symmetry, reduction to the 1-D oracle.
 *
 * Build: gcc -O2 -ffp-contract=off -fopenmp -shared -fPIC (oracle/build.py).  `omp parallel for`
 * over the spatial index is the only parallelism; it does not change any result.
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define REAL double
#define FN(name) name##_f64
#define R_FMA fma
#define R_SQRT sqrt
#define R_FABS fabs
#define R_FMAX fmax
#include "schemes.inc"
#include "heat2d.inc"
#undef REAL
#undef FN
#undef R_FMA
#undef R_SQRT
#undef R_FABS
#undef R_FMAX

#define REAL float
#define FN(name) name##_f32
#define R_FMA fmaf
#define R_SQRT sqrtf
#define R_FABS fabsf
#define R_FMAX fmaxf
#include "schemes.inc"
#include "heat2d.inc"
#undef REAL
#undef FN
#undef R_FMA
#undef R_SQRT
#undef R_FABS
#undef R_FMAX

/* threads the parallel loops will use (reported next to the timed baseline) */
int oracle_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void oracle_set_num_threads(int n) {
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}
