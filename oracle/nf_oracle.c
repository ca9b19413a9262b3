/*
 * nf_oracle.c -- CPU ORACLE for the Abacus near-field force.  TEST INFRASTRUCTURE ONLY.
 *
 * This file is the plain, slow, double-precision statement of what the CUDA path
 * (paper_2110_11392_b200/csrc) must compute.  It is imported only by tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs.  It shares no
 * code, header, table or helper with the CUDA path and the product never calls it.
 *
 * What it follows (reference = /root/reference/PAPER.md, arXiv 2110.11392):
 *   - near-field domain: "every cell interacting with itself and its 124 nearest neighbor
 *     cells (for near-field radius R=2) using open boundary conditions and Newtonian
 *     gravity, or a softened form thereof"            PAPER.md:218 (sec. 3.4.1), :62 (sec. 2.1)
 *   - softening law, Eq. 3: F = [10 - 15u + 6u^2] r/eps_s^3 (u = r/eps_s < 1), r/r^3 else
 *                                                     PAPER.md:132 (sec. 3.2)
 *   - eps_s = 2.16 eps_p                              PAPER.md:143 (sec. 3.2, Fig. 4 caption :141)
 *   - grid of K^3 (=CPD^3) cells, particles kept in grid order, offsets from cell centres
 *                                                     PAPER.md:72 (sec. 2.2), :264 (sec. 3.5.1)
 *   - "handles the periodic wrap" by shifting whole cells (pencil-centred coordinates)
 *                                                     PAPER.md:232 (sec. 3.4.2)
 * Readings where the paper is silent are those of SURVEY.md 8(c) S1-S14, listed in DESIGN.md.
 *
 * The near field is exact by definition (a direct sum), so the oracle IS that definition:
 * piecewise Eq. 3 with a branch (not the GPU's min form), no blocking, no reordering beyond
 * the loop nest "sink cell -> (a,b,c) lexicographic -> sink -> source".
 *
 * Parity pins (tests/test_oracle_pins.py; variants incl. the unsoftened law: tests/test_oracle_variant_pins.py): two-particle closed form inside/outside eps_s,
 * cell-based cutoff, periodic wrap, one-particle-per-cell lattice => 0, momentum sum = 0,
 * all-pairs brute force masked to near-field cell pairs, integer pair-count identity,
 * CPD = 2R+1 => plain all-pairs, whole-cell translation, input-order invariance.
 * Every function below is pinned; nothing here is "parity unpinned".
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define NFO_SPLINE_PER_PLUMMER 2.16 /* eps_s = 2.16 eps_p */

int nfo_max_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* Scalar force law of Eq. 3: returns f such that F = f * r_vec. */
double nfo_force_factor(double r, double eps_s) {
    if (r < eps_s) {
        double u = r / eps_s;
        return (10.0 - 15.0 * u + 6.0 * u * u) / (eps_s * eps_s * eps_s);
    }
    return 1.0 / (r * r * r);
}

/* Plummer law, Eq. 2: f such that F = f * r_vec.  Used only by the pin that
 * checks the 2.16 conversion against "match the small-scale Plummer force". */
double nfo_plummer_factor(double r, double eps_p) {
    double s = r * r + eps_p * eps_p;
    return 1.0 / (s * sqrt(s));
}

/*
 * Binning (PAPER.md:72 grid order; :264 offsets relative to cell centres; reading S5):
 * per axis t = (double)x * (CPD/box); I = floor(t); cell index = I mod CPD (non-negative);
 * offset from the cell centre, in box units, = (t - I - 0.5) * (box/CPD), kept in double.
 * key = (cx*CPD + cy)*CPD + cz  (z fastest).
 * Returns 0, or -1 if a position is not finite.
 */
int nfo_bin(const float *pos, int64_t N, int cpd, double box, int32_t *cell, double *off) {
    const double scale = (double)cpd / box;
    const double cellsz = box / (double)cpd;
    int bad = 0;
    for (int64_t i = 0; i < N; ++i) {
        int c[3];
        for (int k = 0; k < 3; ++k) {
            double x = (double)pos[3 * i + k];
            if (!isfinite(x)) { bad = 1; x = 0.0; }
            double t = x * scale;
            double I = floor(t);
            double m = fmod(I, (double)cpd);
            if (m < 0) m += (double)cpd;
            c[k] = (int)m;
            if (off) off[3 * i + k] = (t - I - 0.5) * cellsz;
        }
        cell[i] = (c[0] * cpd + c[1]) * cpd + c[2];
    }
    return bad ? -1 : 0;
}

/* Grid-ordered lists (CellInfo offset+count :399): stable counting sort of
 * particle indices by cell key; within a cell, ascending original index (reading S12).
 * offsets has ncell+1 entries; order[s] = original index of the s-th particle in grid order. */
void nfo_cell_lists(const int32_t *cell, int64_t N, int64_t ncell, int64_t *offsets, int64_t *order) {
    memset(offsets, 0, (size_t)(ncell + 1) * sizeof(int64_t));
    for (int64_t i = 0; i < N; ++i) offsets[cell[i] + 1]++;
    for (int64_t c = 0; c < ncell; ++c) offsets[c + 1] += offsets[c];
    int64_t *cur = (int64_t *)malloc((size_t)ncell * sizeof(int64_t));
    memcpy(cur, offsets, (size_t)ncell * sizeof(int64_t));
    for (int64_t i = 0; i < N; ++i) order[cur[cell[i]]++] = i;
    free(cur);
}

static inline int wrap_idx(int v, int cpd, int *image) {
    /* v in [-cpd, 2cpd): image = floor(v/cpd) in {-1,0,1} */
    int w = 0;
    if (v < 0) { v += cpd; w = -1; }
    else if (v >= cpd) { v -= cpd; w = 1; }
    *image = w;
    return v;
}

/* Neighbour list of one cell (reading S3): the (2R+1)^3 cells
 * ((i+a) mod CPD, (j+b) mod CPD, (k+c) mod CPD), (a,b,c) in [-R,R]^3 lexicographic (a slowest),
 * each with its periodic image count floor((i+a)/CPD) etc. in {-1,0,1}.  */
void nfo_neighbors(int cpd, int R, int cellid, int32_t *ids, int8_t *image) {
    int k = cellid % cpd, j = (cellid / cpd) % cpd, i = cellid / (cpd * cpd);
    int n = 0;
    for (int a = -R; a <= R; ++a)
        for (int b = -R; b <= R; ++b)
            for (int c = -R; c <= R; ++c) {
                int wa, wb, wc;
                int ia = wrap_idx(i + a, cpd, &wa), jb = wrap_idx(j + b, cpd, &wb), kc = wrap_idx(k + c, cpd, &wc);
                ids[n] = (ia * cpd + jb) * cpd + kc;
                image[3 * n + 0] = (int8_t)wa;
                image[3 * n + 1] = (int8_t)wb;
                image[3 * n + 2] = (int8_t)wc;
                ++n;
            }
}

/* Number of (sink, source) pairs the definition visits, q != p:
 * sum over cells c of n_c * sum over the (2R+1)^3 neighbours c' of n_c', minus N.
 * Counted by walking the same neighbour lists as nfo_accel (not by a closed form). */
int64_t nfo_pair_count(const int64_t *offsets, int cpd, int R) {
    int64_t ncell = (int64_t)cpd * cpd * cpd, total = 0, N = offsets[ncell];
    int nn = (2 * R + 1) * (2 * R + 1) * (2 * R + 1);
#pragma omp parallel
    {
        int32_t *ids = (int32_t *)malloc((size_t)nn * sizeof(int32_t));
        int8_t *img = (int8_t *)malloc((size_t)nn * 3);
#pragma omp for reduction(+ : total) schedule(static)
        for (int64_t c = 0; c < ncell; ++c) {
            int64_t nc = offsets[c + 1] - offsets[c];
            if (nc == 0) continue;
            nfo_neighbors(cpd, R, (int)c, ids, img);
            int64_t s = 0;
            for (int n = 0; n < nn; ++n) s += offsets[ids[n] + 1] - offsets[ids[n]];
            total += nc * s;
        }
        free(ids);
        free(img);
    }
    return total - N;
}

/*
 * Near-field acceleration (the definition):
 *   for each sink cell C=(i,j,k), for (a,b,c) in [-R,R]^3 lexicographic:
 *     S = ((i+a) mod CPD, (j+b) mod CPD, (k+c) mod CPD)
 *     for sink p in C, for source q in S, q != p:
 *        d  = (off_q - off_p) + (a,b,c)*cell          -- x_source - x_sink, cell-pair image (S3, S6)
 *        r2 = d.d ; if r2 == 0 continue               -- F(0) = 0 (S4)
 *        f  = Eq. 3 with eps_s = 2.16 eps_p           -- PAPER.md:132, :143
 *        a_p += gm * f * d                            -- attractive, gm = G*m (S7)
 * sink_cells: list of n_sink_cells cell ids to evaluate, or NULL for all cells.
 * acc[N][3] (double, input order) is written only for particles in evaluated cells; the
 * caller zero-fills.  Returns the number of pairs evaluated (q != p, r2 == 0 included), or
 * -1 on a non-finite position / bad arguments.
 */
int64_t nfo_accel(const float *pos, int64_t N, int cpd, int R, double eps_p, double box, double gm,
                  const int32_t *sink_cells, int64_t n_sink_cells, double *acc, int nthreads) {
    if (N < 0 || R < 1 || cpd < 2 * R + 1 || !(eps_p > 0) || !(box > 0)) return -1;
    const int64_t ncell = (int64_t)cpd * cpd * cpd;
    const double cellsz = box / (double)cpd;
    const double eps_s = NFO_SPLINE_PER_PLUMMER * eps_p;
    const int nn = (2 * R + 1) * (2 * R + 1) * (2 * R + 1);

    int32_t *cell = (int32_t *)malloc((size_t)(N > 0 ? N : 1) * sizeof(int32_t));
    double *off = (double *)malloc((size_t)(N > 0 ? N : 1) * 3 * sizeof(double));
    int64_t *offsets = (int64_t *)malloc((size_t)(ncell + 1) * sizeof(int64_t));
    int64_t *order = (int64_t *)malloc((size_t)(N > 0 ? N : 1) * sizeof(int64_t));
    if (!cell || !off || !offsets || !order) { free(cell); free(off); free(offsets); free(order); return -1; }
    if (nfo_bin(pos, N, cpd, box, cell, off) != 0) { free(cell); free(off); free(offsets); free(order); return -1; }
    nfo_cell_lists(cell, N, ncell, offsets, order);

    /* grid-ordered copy of the offsets so the inner loop streams */
    double *so = (double *)malloc((size_t)(N > 0 ? N : 1) * 3 * sizeof(double));
    for (int64_t s = 0; s < N; ++s) {
        int64_t i = order[s];
        so[3 * s + 0] = off[3 * i + 0]; so[3 * s + 1] = off[3 * i + 1]; so[3 * s + 2] = off[3 * i + 2];
    }

    const int64_t nwork = sink_cells ? n_sink_cells : ncell;
    int64_t pairs = 0;
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
#endif
#pragma omp parallel
    {
        int32_t *ids = (int32_t *)malloc((size_t)nn * sizeof(int32_t));
        int8_t *img = (int8_t *)malloc((size_t)nn * 3);
#pragma omp for schedule(dynamic, 1) reduction(+ : pairs)
        for (int64_t w = 0; w < nwork; ++w) {
            const int C = sink_cells ? sink_cells[w] : (int)w;
            const int64_t p0 = offsets[C], p1 = offsets[C + 1];
            if (p0 == p1) continue;
            nfo_neighbors(cpd, R, C, ids, img);
            for (int64_t p = p0; p < p1; ++p) {
                double ax = 0.0, ay = 0.0, az = 0.0;
                const double px = so[3 * p], py = so[3 * p + 1], pz = so[3 * p + 2];
                int n = 0;
                for (int a = -R; a <= R; ++a)
                    for (int b = -R; b <= R; ++b)
                        for (int c = -R; c <= R; ++c, ++n) {
                            const int S = ids[n];
                            const double sx = a * cellsz, sy = b * cellsz, sz = c * cellsz;
                            const int64_t q0 = offsets[S], q1 = offsets[S + 1];
                            for (int64_t q = q0; q < q1; ++q) {
                                if (q == p) continue;
                                const double dx = (so[3 * q] - px) + sx;
                                const double dy = (so[3 * q + 1] - py) + sy;
                                const double dz = (so[3 * q + 2] - pz) + sz;
                                const double r2 = dx * dx + dy * dy + dz * dz;
                                ++pairs;
                                if (r2 == 0.0) continue;
                                const double r = sqrt(r2);
                                double f;
                                if (r < eps_s) {
                                    const double u = r / eps_s;
                                    f = (10.0 - 15.0 * u + 6.0 * u * u) / (eps_s * eps_s * eps_s);
                                } else {
                                    f = 1.0 / (r2 * r);
                                }
                                ax += gm * f * dx; ay += gm * f * dy; az += gm * f * dz;
                            }
                        }
                const int64_t i = order[p];
                acc[3 * i] = ax; acc[3 * i + 1] = ay; acc[3 * i + 2] = az;
            }
        }
        free(ids);
        free(img);
    }
    free(so); free(cell); free(off); free(offsets); free(order);
    return pairs;
}

/*
 * Variants of the near-field sum the paper configures at build time (Fig. 19:
 * "Near-force softening technique", "Compute FOF-scale density"), same loop nest and cell-pair
 * definition as nfo_accel:
 *   law = 0  spline softening, Eq. 3, eps_s = 2.16 eps_p
 *   law = 1  Plummer softening, Eq. 2: F = r / (r^2 + eps_p^2)^(3/2)
 *   law = 2  no softening: "Newtonian gravity, or a softened form thereof", F = r/|r|^3;
 *            eps_p is ignored; a coincident pair (r = 0) contributes 0, as F(0) = 0 does for
 *            both softened laws (reading S4 carried over; reading N1)
 *   dens_b > 0 and dens != NULL: the FoF-scale density estimate of sec. 3.4.4,
 *       "an apodized top-hat density estimate 1 - r^2/b^2 (for r < b), which is computed as
 *       b^2 - r^2 on the GPU":   dens_p = sum over sources q != p of the same (2R+1)^3 cells
 *       with r < b of (b^2 - r^2), r = |d| the same separation the force uses.
 *       Readings (D1-D3): the particle itself is not counted (q != p, as in the force
 *       loop); a distinct particle at r = 0 counts b^2; the sum is left unnormalised in
 *       (length unit)^2, as the paper's kernel leaves it.
 * acc may be NULL (density only).  Returns pairs visited, or -1.
 */
int64_t nfo_accel_variant(const float *pos, int64_t N, int cpd, int R, double eps_p, double box, double gm, int law, double dens_b,
                          const int32_t *sink_cells, int64_t n_sink_cells, double *acc, double *dens, int nthreads) {
    if (N < 0 || R < 1 || cpd < 2 * R + 1 || !(eps_p > 0) || !(box > 0) || law < 0 || law > 2 || dens_b < 0) return -1;
    const int64_t ncell = (int64_t)cpd * cpd * cpd;
    const double cellsz = box / (double)cpd;
    const double eps_s = NFO_SPLINE_PER_PLUMMER * eps_p;
    const double b2 = dens_b * dens_b;
    const int nn = (2 * R + 1) * (2 * R + 1) * (2 * R + 1);
    int32_t *cell = (int32_t *)malloc((size_t)(N > 0 ? N : 1) * sizeof(int32_t));
    double *off = (double *)malloc((size_t)(N > 0 ? N : 1) * 3 * sizeof(double));
    int64_t *offsets = (int64_t *)malloc((size_t)(ncell + 1) * sizeof(int64_t));
    int64_t *order = (int64_t *)malloc((size_t)(N > 0 ? N : 1) * sizeof(int64_t));
    double *so = (double *)malloc((size_t)(N > 0 ? N : 1) * 3 * sizeof(double));
    if (!cell || !off || !offsets || !order || !so || nfo_bin(pos, N, cpd, box, cell, off) != 0) {
        free(cell); free(off); free(offsets); free(order); free(so);
        return -1;
    }
    nfo_cell_lists(cell, N, ncell, offsets, order);
    for (int64_t s = 0; s < N; ++s) {
        int64_t i = order[s];
        so[3 * s + 0] = off[3 * i + 0]; so[3 * s + 1] = off[3 * i + 1]; so[3 * s + 2] = off[3 * i + 2];
    }
    const int64_t nwork = sink_cells ? n_sink_cells : ncell;
    int64_t pairs = 0;
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
#endif
#pragma omp parallel
    {
        int32_t *ids = (int32_t *)malloc((size_t)nn * sizeof(int32_t));
        int8_t *img = (int8_t *)malloc((size_t)nn * 3);
#pragma omp for schedule(dynamic, 1) reduction(+ : pairs)
        for (int64_t w = 0; w < nwork; ++w) {
            const int C = sink_cells ? sink_cells[w] : (int)w;
            const int64_t p0 = offsets[C], p1 = offsets[C + 1];
            if (p0 == p1) continue;
            nfo_neighbors(cpd, R, C, ids, img);
            for (int64_t p = p0; p < p1; ++p) {
                double ax = 0.0, ay = 0.0, az = 0.0, wd = 0.0;
                const double px = so[3 * p], py = so[3 * p + 1], pz = so[3 * p + 2];
                int n = 0;
                for (int a = -R; a <= R; ++a)
                    for (int b = -R; b <= R; ++b)
                        for (int c = -R; c <= R; ++c, ++n) {
                            const int S = ids[n];
                            const double sx = a * cellsz, sy = b * cellsz, sz = c * cellsz;
                            const int64_t q0 = offsets[S], q1 = offsets[S + 1];
                            for (int64_t q = q0; q < q1; ++q) {
                                if (q == p) continue;
                                const double dx = (so[3 * q] - px) + sx;
                                const double dy = (so[3 * q + 1] - py) + sy;
                                const double dz = (so[3 * q + 2] - pz) + sz;
                                const double r2 = dx * dx + dy * dy + dz * dz;
                                ++pairs;
                                if (r2 < b2) wd += b2 - r2;
                                if (r2 == 0.0) continue;                 /* F(0) = 0 for both laws */
                                double f;
                                if (law == 1) {
                                    const double s2 = r2 + eps_p * eps_p;    /* Eq. 2 */
                                    f = 1.0 / (s2 * sqrt(s2));
                                } else if (law == 2) {
                                    f = 1.0 / (r2 * sqrt(r2));               /* Newtonian */
                                } else {
                                    const double r = sqrt(r2);
                                    if (r < eps_s) {
                                        const double u = r / eps_s;          /* Eq. 3 */
                                        f = (10.0 - 15.0 * u + 6.0 * u * u) / (eps_s * eps_s * eps_s);
                                    } else {
                                        f = 1.0 / (r2 * r);
                                    }
                                }
                                ax += gm * f * dx; ay += gm * f * dy; az += gm * f * dz;
                            }
                        }
                const int64_t i = order[p];
                if (acc) { acc[3 * i] = ax; acc[3 * i + 1] = ay; acc[3 * i + 2] = az; }
                if (dens) dens[i] = wd;
            }
        }
        free(ids);
        free(img);
    }
    free(so); free(cell); free(off); free(offsets); free(order);
    return pairs;
}

/*
 * Cell multipoles, Eq. 4 (sec. 3.3.2), in the complete basis of
 * cml = (p+3)(p+2)(p+1)/6 values per cell:
 *     M_{i,j,k}^{a,b,c} = sum_q x_q^a y_q^b z_q^c,   0 <= a <= p, 0 <= b <= p-a, 0 <= c <= p-a-b,
 * (x_q, y_q, z_q) = displacement of particle q "from the origin of cell (i,j,k)" = its offset from
 * the cell centre (nfo_bin, reading S5), in length units.  The loop nest is the paper's pseudo-code
 * (garbled in the extraction; restored from Eq. 4): for each particle, mx runs over
 * x^a, mxy over x^a y^b, mxyz over x^a y^b z^c by repeated multiplication, and M[a,b,c] += mxyz with
 * (a,b,c) in that nesting order, which is also the order of the output index.
 * M: ncell * cml doubles, cell-major (key = (cx*CPD+cy)*CPD+cz).  Particles of a cell are added in
 * ascending input order.  Returns cml, or -1.
 */
int nfo_multipoles(const float *pos, int64_t N, int cpd, double box, int order, double *M) {
    if (N < 0 || cpd < 1 || !(box > 0) || order < 0 || order > 16) return -1;
    const int cml = (order + 3) * (order + 2) * (order + 1) / 6;
    const int64_t ncell = (int64_t)cpd * cpd * cpd;
    int32_t *cell = (int32_t *)malloc((size_t)(N > 0 ? N : 1) * sizeof(int32_t));
    double *off = (double *)malloc((size_t)(N > 0 ? N : 1) * 3 * sizeof(double));
    if (!cell || !off || nfo_bin(pos, N, cpd, box, cell, off) != 0) { free(cell); free(off); return -1; }
    memset(M, 0, (size_t)ncell * cml * sizeof(double));
    for (int64_t q = 0; q < N; ++q) {
        double *Mc = M + (size_t)cell[q] * cml;
        const double X = off[3 * q], Y = off[3 * q + 1], Z = off[3 * q + 2];
        int idx = 0;
        double mx = 1.0;
        for (int a = 0; a <= order; ++a) {
            double mxy = mx;
            for (int b = 0; b <= order - a; ++b) {
                double mxyz = mxy;
                for (int c = 0; c <= order - a - b; ++c) {
                    Mc[idx++] += mxyz;
                    mxyz *= Z;
                }
                mxy *= Y;
            }
            mx *= X;
        }
    }
    free(cell); free(off);
    return cml;
}

/*
 * Kick and Drift of the KDK leapfrog (sec. 3.1 "standard second-order leapfrog
 * Kick-Drift-Kick"; Table 1: Kick "update velocity from t-1/2 to t+1/2", Drift
 * "update position from t to t+1"), on float32 state as the paper stores it:
 *     v <- v + a * dt_kick        x <- x + v_new * dt_drift, wrapped periodically into [0, box)
 * Readings (K1-K3): each update is evaluated in double from the float32 inputs (one
 * product, one sum, separately rounded) and rounded to float32 once; the wrap is
 * w = x - floor(x / box) * box, a result that rounds to box is folded to 0; dt_kick and dt_drift
 * are plain time intervals (the cosmological drift/kick factors are the caller's).
 * No fused multiply-add here, so that the CUDA path can reproduce it bit for bit.
 */
__attribute__((optimize("fp-contract=off")))
void nfo_kick_drift(float *pos, float *vel, const float *acc, int64_t N, double dt_kick, double dt_drift, double box) {
    for (int64_t i = 0; i < 3 * N; ++i) {
        const double prod = (double)acc[i] * dt_kick;
        const float v = (float)((double)vel[i] + prod);
        vel[i] = v;
        const double step = (double)v * dt_drift;
        double x = (double)pos[i] + step;
        const double k = floor(x / box);
        const double back = k * box;
        x = x - back;
        if (x < 0.0) x = 0.0;
        float xf = (float)x;
        if (!(xf < (float)box)) xf = 0.0f;
        pos[i] = xf;
    }
}

/*
 * The particle-dependent part of the time-step criterion, Eq. 1:
 *     max( min over cells c of [v_rms / a_max]_c ,  v_rms,global / a_max,global )
 * v_rms = sqrt(mean |v|^2) "computed without subtracting off the mean velocity",
 * a_max = max |a|, both over the particles of a cell (cells of the CPD^3 grid, binning of nfo_bin)
 * or of the whole box.  Empty cells and cells with a_max = 0 do not constrain the step.
 * out[0] = min_c [v_rms/a_max]_c (+inf if no cell constrains), out[1] = v_rms,global / a_max,global,
 * out[2] = v_rms,global, out[3] = a_max,global.  Returns 0, or -1.
 */
int nfo_timestep_ratio(const float *pos, const float *vel, const float *acc, int64_t N, int cpd, double box, double *out) {
    if (N < 0 || cpd < 1 || !(box > 0)) return -1;
    const int64_t ncell = (int64_t)cpd * cpd * cpd;
    int32_t *cell = (int32_t *)malloc((size_t)(N > 0 ? N : 1) * sizeof(int32_t));
    double *v2 = (double *)calloc((size_t)ncell, sizeof(double));
    double *a2 = (double *)calloc((size_t)ncell, sizeof(double));
    int64_t *cnt = (int64_t *)calloc((size_t)ncell, sizeof(int64_t));
    if (!cell || !v2 || !a2 || !cnt || nfo_bin(pos, N, cpd, box, cell, NULL) != 0) { free(cell); free(v2); free(a2); free(cnt); return -1; }
    double gv2 = 0.0, ga2 = 0.0;
    for (int64_t i = 0; i < N; ++i) {
        const double vx = vel[3 * i], vy = vel[3 * i + 1], vz = vel[3 * i + 2];
        const double ax = acc[3 * i], ay = acc[3 * i + 1], az = acc[3 * i + 2];
        const double s = vx * vx + vy * vy + vz * vz, t = ax * ax + ay * ay + az * az;
        v2[cell[i]] += s; cnt[cell[i]]++;
        if (t > a2[cell[i]]) a2[cell[i]] = t;
        gv2 += s;
        if (t > ga2) ga2 = t;
    }
    double best = INFINITY;
    for (int64_t c = 0; c < ncell; ++c) {
        if (cnt[c] == 0 || a2[c] == 0.0) continue;
        const double r = sqrt(v2[c] / (double)cnt[c]) / sqrt(a2[c]);
        if (r < best) best = r;
    }
    out[0] = best;
    out[2] = N > 0 ? sqrt(gv2 / (double)N) : 0.0;
    out[3] = sqrt(ga2);
    out[1] = ga2 > 0.0 ? out[2] / out[3] : INFINITY;
    free(cell); free(v2); free(a2); free(cnt);
    return 0;
}

/*
 * Taylor evaluation of the far field ("evaluating the force from the resulting Taylor
 * series of the potential in every cell"; "the output is a 3-vector of acceleration for
 * every particle ... about 3 times more floating-point work").  The paper does not print the
 * series; reading (F1): the cell's Taylors are the coefficients T^{a,b,c} of the potential
 * in the same complete basis and index order as the multipoles,
 *     phi(x,y,z) = sum_{a+b+c <= p} T^{a,b,c} x^a y^b z^c,   (x,y,z) = offset from the cell centre,
 * (any factorials are folded into T by whoever produces it), and the far-field acceleration is
 *     a = -grad phi = -( sum a T x^(a-1) y^b z^c,  sum b T x^a y^(b-1) z^c,  sum c T x^a y^b z^(c-1) ).
 * T: ncell * cml doubles, cell-major.  acc[N][3] double, input order.  Returns 0, or -1.
 */
int nfo_taylor_accel(const float *pos, int64_t N, int cpd, double box, int order, const double *T, double *acc) {
    if (N < 0 || cpd < 1 || !(box > 0) || order < 0 || order > 16) return -1;
    const int cml = (order + 3) * (order + 2) * (order + 1) / 6;
    int32_t *cell = (int32_t *)malloc((size_t)(N > 0 ? N : 1) * sizeof(int32_t));
    double *off = (double *)malloc((size_t)(N > 0 ? N : 1) * 3 * sizeof(double));
    if (!cell || !off || nfo_bin(pos, N, cpd, box, cell, off) != 0) { free(cell); free(off); return -1; }
    for (int64_t q = 0; q < N; ++q) {
        const double *Tc = T + (size_t)cell[q] * cml;
        const double X = off[3 * q], Y = off[3 * q + 1], Z = off[3 * q + 2];
        double xp[18], yp[18], zp[18];
        xp[0] = yp[0] = zp[0] = 1.0;
        for (int k = 1; k <= order; ++k) { xp[k] = xp[k - 1] * X; yp[k] = yp[k - 1] * Y; zp[k] = zp[k - 1] * Z; }
        double gx = 0.0, gy = 0.0, gz = 0.0;
        int idx = 0;
        for (int a = 0; a <= order; ++a)
            for (int b = 0; b <= order - a; ++b)
                for (int c = 0; c <= order - a - b; ++c, ++idx) {
                    const double t = Tc[idx];
                    if (a > 0) gx += t * a * xp[a - 1] * yp[b] * zp[c];
                    if (b > 0) gy += t * b * xp[a] * yp[b - 1] * zp[c];
                    if (c > 0) gz += t * c * xp[a] * yp[b] * zp[c - 1];
                }
        acc[3 * q] = -gx; acc[3 * q + 1] = -gy; acc[3 * q + 2] = -gz;
    }
    free(cell); free(off);
    return 0;
}
