/*
 * ts_oracle.c -- CPU ORACLE for the second-order Trotter-Suzuki lattice step.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT PRODUCT CODE.  Only tests/, the smoke check in
 * __graft_entry__.py and bench.py's cpu_baseline / --impl reference legs may build, link or
 * call it.  It shares no code, header, table or helper with the CUDA library under
 * paper_1208_2407_b200/csrc/ and neither includes the other.
 *
 * It is the algorithm of the paper written out step by step in double precision, in the
 * paper's order, with no blocking, fusion or reordering (PAPER.md = /root/reference/PAPER.md):
 *
 *   - H = H0 + H1 + H2: diagonal + even pairs + odd pairs           PAPER.md:61-77  (Sec. 2)
 *   - exp of each pair block is the 2x2 plane rotation M             PAPER.md:79-81  (Sec. 2)
 *   - U1 = e^{-i dt H0} e^{-i dt H1} e^{-i dt H2}                    PAPER.md:85     (Sec. 2)
 *   - U2 = U1^T U1 (symmetrised, second order)                       PAPER.md:87-89  (Eq. 3)
 *   - 2-D: diagonal + two parts per dimension                        PAPER.md:91-93  (Sec. 2)
 *   - norm of the state                                              PAPER.md:49     (Sec. 2)
 *
 * Readings of the paper where it is silent or garbled:
 *   R1 the pair block is [[a, +i b],[+i b, a]] with a signed, caller-supplied b;
 *   R2 U2(dt) = U1^T(dt/2) U1(dt/2): outer stages use the half angle;
 *   R3 without a potential the innermost kinetic part (vertical-odd) gets one full-angle
 *      sweep; with a potential the phase sits at the centre between two half sweeps;
 *   R5 order, outermost to innermost: X-even, X-odd, Y-even, Y-odd;
 *   R6 even pairs are (2k, 2k+1), odd pairs are (2k+1, 2k+2), 0-based;
 *   R7 closed: pairs crossing the edge are omitted and unpaired sites are unchanged;
 *      periodic: the wrap pair (n-1, 0) belongs to the odd sweep (n even);
 *   R10 both outputs of a pair are computed from the OLD values of both inputs.
 *
 * Parity pins (tests/test_oracle_pins.py, none of them re-types this file's formulae):
 * 2-site closed form, dense expm of every part, dense ordered product of a full step,
 * reversibility, dt^2 convergence to exp(-iHt), X/Y commutation, periodic eigenstates,
 * golden tables G1/G2 regenerated from dense matrices.  Nothing here is "parity unpinned".
 *
 * Layout: two planes re[ny][nx], im[ny][nx] of double, x fastest (index y*nx + x).
 * The only parallelism is an optional OpenMP "for" over the independent lines of one sweep
 * (pairs of one sweep are disjoint), enabled with -fopenmp.
 */
#include <stddef.h>
#include <stdint.h>

#ifdef _OPENMP
#include <omp.h>
#endif

/* (psi_p, psi_q) <- M (psi_p, psi_q),  M = [[a, i b],[i b, a]]   PAPER.md:79-81, reading R1/R10 */
static void rotate_pair(double *re, double *im, size_t p, size_t q, double a, double b)
{
    const double rp = re[p], ip = im[p], rq = re[q], iq = im[q];
    /* a*psi_p + i*b*psi_q :  re = a*rp - b*iq,  im = a*ip + b*rq */
    re[p] = a * rp - b * iq;
    im[p] = a * ip + b * rq;
    re[q] = a * rq - b * ip;
    im[q] = a * iq + b * rp;
}

/*
 * One checkerboard sweep.  axis 0 = horizontal (x), axis 1 = vertical (y); parity 0 = even pairs
 * (2k,2k+1), parity 1 = odd pairs (2k+1,2k+2) plus the wrap pair (n-1,0) when periodic.
 * H1 / H2 of PAPER.md:71-77 along one axis, for every line of the lattice.
 */
void oracle_sweep(double *re, double *im, int64_t nx, int64_t ny,
                  int axis, int parity, double a, double b, int periodic)
{
    if (axis == 0) {
#ifdef _OPENMP
#pragma omp parallel for schedule(static)
#endif
        for (int64_t y = 0; y < ny; ++y) {
            for (int64_t x = parity; x + 1 <= nx - 1; x += 2)
                rotate_pair(re, im, (size_t)(y * nx + x), (size_t)(y * nx + x + 1), a, b);
            if (periodic && parity == 1)
                rotate_pair(re, im, (size_t)(y * nx + nx - 1), (size_t)(y * nx), a, b);
        }
    } else {
#ifdef _OPENMP
#pragma omp parallel for schedule(static)
#endif
        for (int64_t x = 0; x < nx; ++x) {
            for (int64_t y = parity; y + 1 <= ny - 1; y += 2)
                rotate_pair(re, im, (size_t)(y * nx + x), (size_t)((y + 1) * nx + x), a, b);
            if (periodic && parity == 1)
                rotate_pair(re, im, (size_t)((ny - 1) * nx + x), (size_t)x, a, b);
        }
    }
}

/* psi(x,y) <- psi(x,y) * (pr + i pi): e^{-i dt H0}, H0 diagonal. */
void oracle_phase(double *re, double *im, int64_t nx, int64_t ny,
                  const double *pot_re, const double *pot_im)
{
#ifdef _OPENMP
#pragma omp parallel for schedule(static)
#endif
    for (int64_t y = 0; y < ny; ++y)
        for (int64_t x = 0; x < nx; ++x) {
            const size_t i = (size_t)(y * nx + x);
            const double r = re[i], m = im[i];
            re[i] = r * pot_re[i] - m * pot_im[i];
            im[i] = r * pot_im[i] + m * pot_re[i];
        }
}

/* One second-order step U2, Eq. 3 with readings R2, R3, R5. */
void oracle_step(double *re, double *im, int64_t nx, int64_t ny,
                 double a_half, double b_half, double a_full, double b_full,
                 const double *pot_re, const double *pot_im, int periodic)
{
    oracle_sweep(re, im, nx, ny, 0, 0, a_half, b_half, periodic);      /* X even, half */
    oracle_sweep(re, im, nx, ny, 0, 1, a_half, b_half, periodic);      /* X odd,  half */
    oracle_sweep(re, im, nx, ny, 1, 0, a_half, b_half, periodic);      /* Y even, half */
    if (pot_re == NULL) {
        oracle_sweep(re, im, nx, ny, 1, 1, a_full, b_full, periodic);  /* Y odd,  full */
    } else {
        oracle_sweep(re, im, nx, ny, 1, 1, a_half, b_half, periodic);  /* Y odd,  half */
        oracle_phase(re, im, nx, ny, pot_re, pot_im);                  /* potential    */
        oracle_sweep(re, im, nx, ny, 1, 1, a_half, b_half, periodic);  /* Y odd,  half */
    }
    oracle_sweep(re, im, nx, ny, 1, 0, a_half, b_half, periodic);      /* Y even, half */
    oracle_sweep(re, im, nx, ny, 0, 1, a_half, b_half, periodic);      /* X odd,  half */
    oracle_sweep(re, im, nx, ny, 0, 0, a_half, b_half, periodic);      /* X even, half */
}

/* n_steps applications of U2.  pot_re/pot_im NULL => no potential. */
void oracle_evolve(double *re, double *im, int64_t nx, int64_t ny,
                   double a_half, double b_half, double a_full, double b_full,
                   const double *pot_re, const double *pot_im,
                   int periodic, int64_t n_steps)
{
    for (int64_t s = 0; s < n_steps; ++s)
        oracle_step(re, im, nx, ny, a_half, b_half, a_full, b_full, pot_re, pot_im, periodic);
}

/* sum |psi|^2, plain left-to-right double sum with Kahan compensation. */
double oracle_norm2(const double *re, const double *im, int64_t nx, int64_t ny)
{
    double sum = 0.0, comp = 0.0;
    const size_t n = (size_t)nx * (size_t)ny;
    for (size_t i = 0; i < n; ++i) {
        const double term = re[i] * re[i] + im[i] * im[i] - comp;
        const double t = sum + term;
        comp = (t - sum) - term;
        sum = t;
    }
    return sum;
}

/* threads the OpenMP loops will use (1 without OpenMP); reported by bench.py as "cores" */
int oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void oracle_set_num_threads(int n)
{
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}
