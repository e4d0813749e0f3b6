/*
 * ORACLE -- TEST INFRASTRUCTURE ONLY.
 *
 * Plain, slow, obviously-correct CPU implementation of what the CUDA hot path
 * computes: the staggered Dirac hopping operator of Eq. (1) (PAPER.md:49-54,
 * Sec. 4.2), the even-odd preconditioned normal operator M = m^2 - D_eo D_oe
 * (BASELINE.json north_star) and Conjugate Gradient on it.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
 * reference legs may build, load or call this.  It shares no code, header,
 * table or helper with paper_2502_03249_b200/ (the CUDA product), and the product
 * never falls back to it.
 *
 * Deliberately naive: AoS, full-lattice lexicographic indexing, explicit
 * coordinate loops, C99 complex arithmetic, OpenMP over sites and nothing
 * cleverer.  No blocking, no even/odd compaction, no sign tables.
 *
 * What pins it (tests/test_oracle_pins.py, all `-m "not gpu"`):
 *   anti-hermiticity D_oe = -D_eo^dagger, M hermitian positive definite, the
 *   free-field plane-wave spectrum m^2 + 4 sum sin^2 p_mu (periodic space,
 *   antiperiodic time), the pointwise free-field closed form, the constant-field
 *   seam test, the hand-derived point-source sign table (tests/golden/), gauge
 *   covariance, a dense 384x384 brute-force solve at 4^4, CG finite termination
 *   on the 4-eigenvalue free field, the large-mass limit.
 * Parity unpinned (self-consistency only): the exact fp64 iteration count on
 *   random links, and the residual the fp32 CG variant attains.
 *
 * Build: gcc -O2 -fopenmp -fcx-limited-range -shared -fPIC (oracle/__init__.py).
 */
#include <complex.h>
#include <math.h>

/* lexicographic index, x0 fastest (N_sigma^3 x N_tau; mu = 3 is time) */
static long lex_index(const int N[4], const int x[4])
{
    return (long)x[0] + (long)N[0] * ((long)x[1] + (long)N[1] * ((long)x[2] + (long)N[2] * (long)x[3]));
}

static int site_parity(const int x[4]) { return (x[0] + x[1] + x[2] + x[3]) & 1; }

static int index_parity(const int N[4], long i)
{
    int x[4];
    x[0] = (int)(i % N[0]); i /= N[0];
    x[1] = (int)(i % N[1]); i /= N[1];
    x[2] = (int)(i % N[2]); i /= N[2];
    x[3] = (int)i;
    return site_parity(x);
}

/* Kogut-Susskind phase eta_mu(x) = (-1)^{x_0 + ... + x_{mu-1}}  (configs[0]) */
static int ks_phase(int mu, const int x[4])
{
    int s = 0;
    for (int nu = 0; nu < mu; ++nu) s += x[nu];
    return (s & 1) ? -1 : +1;
}

#define REAL double
#define SFX f64
#define CONJ conj
#define CREAL creal
#define CIMAG cimag
#include "staggered_impl.inc"
#undef REAL
#undef SFX
#undef CONJ
#undef CREAL
#undef CIMAG

#define REAL float
#define SFX f32
#define CONJ conjf
#define CREAL crealf
#define CIMAG cimagf
#include "staggered_impl.inc"
#undef REAL
#undef SFX
#undef CONJ
#undef CREAL
#undef CIMAG

#ifdef _OPENMP
#include <omp.h>
int oracle_num_threads(void) { return omp_get_max_threads(); }
void oracle_set_num_threads(int n) { omp_set_num_threads(n); }
#else
int oracle_num_threads(void) { return 1; }
void oracle_set_num_threads(int n) { (void)n; }
#endif
