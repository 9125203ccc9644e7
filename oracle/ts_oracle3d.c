/*
 * ts_oracle3d.c -- CPU ORACLE for the second-order Trotter-Suzuki step on a THREE-dimensional
 * lattice (the extension the paper names as its next direction, Sec. 5).
 *
 * THIS IS TEST INFRASTRUCTURE, NOT PRODUCT CODE.  Only tests/, the smoke check in
 * __graft_entry__.py and bench.py's cpu_baseline / --impl reference legs may build, link or
 * call it.  It shares no code, header, table or helper with the CUDA library under
 * paper_1208_2407_b200/csrc/ (nor with ts_oracle.c, the 2-D oracle, which stays as it was
 * first committed) and neither includes the other.
 *
 * What it computes.  "Extending the algorithm for more than one dimension is also
 * straightforward, as we can simply perform a decomposition of the Hamiltonian into [...] the
 * diagonal energies, and two terms for each dimension": in three dimensions
 * that is seven parts -- H0 (diagonal) and an even-pair and an odd-pair part along x, y and z
 * (PAPER.md:71-77 per axis) -- each pair part exponentiated exactly by the 2x2 rotation
 * M = [[a, i b],[i b, a]], composed as U1 = e^{H0} e^{..} .. and symmetrised,
 * U2 = U1^T U1 (Eq. 3).  Written out, in double precision, in that order, with
 * no blocking, fusion or reordering:
 *
 *   Xe(h) Xo(h) Ye(h) Yo(h) Ze(h) [ Zo(f) | Zo(h) P Zo(h) ] Ze(h) Yo(h) Ye(h) Xo(h) Xe(h)
 *
 * Readings (the 2-D ones carried over; R14 is new):
 *   R1  the pair block is [[a, +i b],[+i b, a]], b signed and caller-supplied;
 *   R2  outer stages use the half angle;
 *   R3  without a potential the innermost kinetic part (z-odd) gets one full-angle sweep; with a
 *       potential the phase P sits at the centre between two z-odd half sweeps;
 *   R6  even pairs (2k, 2k+1), odd pairs (2k+1, 2k+2), 0-based, per axis;
 *   R7  per-axis boundary: closed = pairs crossing the edge omitted, periodic = the wrap pair
 *       (n-1, 0) belongs to the odd sweep (n even);
 *   R10 both outputs of a pair come from the OLD values of both inputs;
 *   R14 order of the six kinetic parts, outermost to innermost: Xe, Xo, Ye, Yo, Ze, Zo (the 2-D
 *       order R5 with the new axis innermost).  Sweeps along different axes commute, so only
 *       the position of P (after all six, at the centre) and even-before-odd per axis matter.
 *
 * Parity pins (tests/test_oracle_3d.py; none re-types this file's formulae): every sweep against
 * dense expm(i theta A_part) on small lattices, the full step against the ordered dense product,
 * reduction to the pinned 2-D oracle when nz = 1 (and when nx = 1 with axes renamed),
 * reversibility, dt^2 convergence to expm(-iHT), norm conservation, periodic +-1 eigenstates in
 * closed form, constant potential = global phase.  Nothing here is "parity unpinned".
 *
 * Layout: planes re[nz][ny][nx], im[nz][ny][nx] of double, x fastest: index (z*ny + y)*nx + x.
 * The only parallelism is an optional OpenMP "for" over independent lines of one sweep.
 */
#include <stddef.h>
#include <stdint.h>

/* (psi_p, psi_q) <- [[a, i b],[i b, a]] (psi_p, psi_q) */
static void rotate_pair3(double *re, double *im, size_t p, size_t q, double a, double b)
{
    const double rp = re[p], ip = im[p], rq = re[q], iq = im[q];
    re[p] = a * rp - b * iq;
    im[p] = a * ip + b * rq;
    re[q] = a * rq - b * ip;
    im[q] = a * iq + b * rp;
}

/*
 * One checkerboard sweep along `axis` (0 = x, 1 = y, 2 = z): parity 0 = pairs (2k, 2k+1),
 * parity 1 = pairs (2k+1, 2k+2) plus the wrap pair (n-1, 0) if that axis is periodic; for every
 * line of the lattice along that axis.  H1 / H2 of PAPER.md:71-77 per dimension.
 */
void oracle3_sweep(double *re, double *im, int64_t nx, int64_t ny, int64_t nz,
                   int axis, int parity, double a, double b, int periodic)
{
    /* a line along `axis` starts at (u, v) in the other two coordinates */
    const int64_t n = axis == 0 ? nx : (axis == 1 ? ny : nz);
    const int64_t stride = axis == 0 ? 1 : (axis == 1 ? nx : nx * ny);
    const int64_t nu = axis == 0 ? ny : nx;              /* faster of the other two */
    const int64_t nv = axis == 2 ? ny : nz;              /* slower of the other two */
    const int64_t su = axis == 0 ? nx : 1;
    const int64_t sv = axis == 2 ? nx : nx * ny;
#ifdef _OPENMP
#pragma omp parallel for schedule(static)
#endif
    for (int64_t v = 0; v < nv; ++v)
        for (int64_t u = 0; u < nu; ++u) {
            const int64_t base = v * sv + u * su;
            for (int64_t i = parity; i + 1 <= n - 1; i += 2)
                rotate_pair3(re, im, (size_t)(base + i * stride), (size_t)(base + (i + 1) * stride), a, b);
            if (periodic && parity == 1)
                rotate_pair3(re, im, (size_t)(base + (n - 1) * stride), (size_t)base, a, b);
        }
}

/* psi <- psi * (pr + i pi) at every site: e^{-i dt H0}, H0 diagonal. */
void oracle3_phase(double *re, double *im, int64_t n_sites, const double *pot_re, const double *pot_im)
{
#ifdef _OPENMP
#pragma omp parallel for schedule(static)
#endif
    for (int64_t i = 0; i < n_sites; ++i) {
        const double r = re[i], m = im[i];
        re[i] = r * pot_re[i] - m * pot_im[i];
        im[i] = r * pot_im[i] + m * pot_re[i];
    }
}

/* One second-order step in 3-D (Eq. 3; readings R2, R3, R14).
 * per[0..2] = periodic flag of the x, y, z axis. */
void oracle3_step(double *re, double *im, int64_t nx, int64_t ny, int64_t nz,
                  double a_half, double b_half, double a_full, double b_full,
                  const double *pot_re, const double *pot_im, const int *per)
{
    oracle3_sweep(re, im, nx, ny, nz, 0, 0, a_half, b_half, per[0]);      /* X even, half */
    oracle3_sweep(re, im, nx, ny, nz, 0, 1, a_half, b_half, per[0]);      /* X odd,  half */
    oracle3_sweep(re, im, nx, ny, nz, 1, 0, a_half, b_half, per[1]);      /* Y even, half */
    oracle3_sweep(re, im, nx, ny, nz, 1, 1, a_half, b_half, per[1]);      /* Y odd,  half */
    oracle3_sweep(re, im, nx, ny, nz, 2, 0, a_half, b_half, per[2]);      /* Z even, half */
    if (pot_re == NULL) {
        oracle3_sweep(re, im, nx, ny, nz, 2, 1, a_full, b_full, per[2]);  /* Z odd,  full */
    } else {
        oracle3_sweep(re, im, nx, ny, nz, 2, 1, a_half, b_half, per[2]);  /* Z odd,  half */
        oracle3_phase(re, im, nx * ny * nz, pot_re, pot_im);              /* potential    */
        oracle3_sweep(re, im, nx, ny, nz, 2, 1, a_half, b_half, per[2]);  /* Z odd,  half */
    }
    oracle3_sweep(re, im, nx, ny, nz, 2, 0, a_half, b_half, per[2]);      /* Z even, half */
    oracle3_sweep(re, im, nx, ny, nz, 1, 1, a_half, b_half, per[1]);      /* Y odd,  half */
    oracle3_sweep(re, im, nx, ny, nz, 1, 0, a_half, b_half, per[1]);      /* Y even, half */
    oracle3_sweep(re, im, nx, ny, nz, 0, 1, a_half, b_half, per[0]);      /* X odd,  half */
    oracle3_sweep(re, im, nx, ny, nz, 0, 0, a_half, b_half, per[0]);      /* X even, half */
}

void oracle3_evolve(double *re, double *im, int64_t nx, int64_t ny, int64_t nz,
                    double a_half, double b_half, double a_full, double b_full,
                    const double *pot_re, const double *pot_im, const int *per, int64_t n_steps)
{
    for (int64_t s = 0; s < n_steps; ++s)
        oracle3_step(re, im, nx, ny, nz, a_half, b_half, a_full, b_full, pot_re, pot_im, per);
}
