/*
 * sr_oracle.c -- CPU oracle for HACC's short-range force path.  TEST INFRASTRUCTURE ONLY.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may load this.  It shares no code, header, table or constant with the CUDA path under
 * paper_1410_2805_b200/csrc and neither includes the other.
 *
 * Everything is plain FP64 on the float32 inputs promoted to double, written from the paper
 * (PAPER.md = /root/reference/PAPER.md, arxiv 1410.2805):
 *
 *   - Eq. 8  (section 2.4): fitted grid force f_grid(r).
 *   - Eq. 12 (section 3.1): f_SR(s) = (s+eps)^(-3/2) - f_grid(s),
 *     s = r.r, f_grid(s) "a 5-th order polynomial in s", eps Plummer softening.
 *   - PAPER.md:175: below the force-matching scale r_s the short-range force is the exact
 *     Newtonian force minus the residual filtered grid force; above it, nothing.
 *   - PAPER.md:201, 362: chaining mesh; only the 27 nearest cells need to be searched.
 *   - PAPER.md:205: kick map (velocity updated with the force, position unchanged) and
 *     stream map (position drifted with the velocity).
 *
 * The method reaches the plain definition exactly (a mesh with cell width >= r_max visits a
 * superset of the in-cutoff pairs once each), so the oracle IS the definition:
 *
 *   a_i = sum_{j != i, s_ij < r_max^2}  m_j * d_ij * [ (s_ij+eps)^(-3/2) - P(s_ij) ],
 *   d_ij = minimum image of (x_j - x_i) in [0,L)^3,  s_ij = d_ij . d_ij,
 *   P(s) = c0 + c1 s + ... + c5 s^5,            n_i = #{ j != i : s_ij < r_max^2 }.
 *
 * Readings of silent points: strict cutoff s < r_max^2 (S9); j == i
 * excluded, coincident distinct particles count and add zero force (S8); minimum image by
 * d >= L/2 -> d -= L, d < -L/2 -> d += L (S10); P multiplies the separation VECTOR, i.e.
 * P(s) ~ f_grid(sqrt s)/sqrt s (S2); only the Newtonian term is softened (S7); G = 1 (S6).
 *
 * Out-of-box inputs: the oracle expects positions in [0, L).  oracle_mesh / cell_coord CLAMP a
 * coordinate outside the box to the first / last cell, whereas the CUDA path WRAPS it (reading
 * S16: x - L floor(x/L)).  That difference is deliberate: tests that feed out-of-box positions
 * to the CUDA path wrap them for the oracle first, through oracle_drift(dt = 0), which is the
 * wrap rule written out.  Do not "fix" either side to match the other.
 *
 * Pins (tests/test_oracle_pins.py): two-particle closed form, cutoff strictness, cubic-lattice
 * neighbour count 92 and zero force, Newton's third law, permutation/translation invariance,
 * brute force == linked-list cell list, Plummer-only reduction vs numpy, Eq. 8 values.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

int oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* Eq. 8, with the constants of PAPER.md:181. */
double oracle_fgrid_eq8(double r)
{
    const double b = 0.72, c = 0.01, d = 0.27, e = 0.0001, f = 360.0, g = 100.0, h = 0.67,
                 l = 17.0;
    double r2 = r * r;
    double ch = cosh(b * r);
    return tanh(b * r) / r2 - b / (r * ch * ch) + c * r * (1.0 + d * r2) * exp(-d * r2) +
           e * (1.0 + f * r2 + g * r2 * r2 + l * r2 * r2 * r2) * exp(-h * r2);
}

/* P(s) = sum c_k s^k, plain power sum (no Horner: written as the definition). */
static double poly5(double s, const double c[6])
{
    double p = 0.0, sk = 1.0;
    for (int k = 0; k < 6; ++k) {
        p += c[k] * sk;
        sk *= s;
    }
    return p;
}

/* Eq. 12. */
double oracle_fsr(double s, double eps, const double c[6])
{
    return pow(s + eps, -1.5) - poly5(s, c);
}

/* Minimum image (reading S10). */
static inline double min_image(double d, double L)
{
    if (d >= 0.5 * L) d -= L;
    else if (d < -0.5 * L) d += L;
    return d;
}

/*
 * Brute force, O(ntargets * n).  targets == NULL -> all particles (ntargets ignored, = n).
 * Outputs (length ntargets): ax, ay, az in double; nbr = n_i.  Returns C = sum n_i over the
 * targets computed.  min_gap (may be NULL) receives min |s - r_max^2| / r_max^2 over all
 * tested pairs, so a caller can assert no pair sits within rounding of the cutoff (S11).
 */
uint64_t oracle_sr_brute(int64_t n, const float *x, const float *y, const float *z,
                         const float *m, double L, float r_max, float eps_f,
                         const float poly_f[6], int64_t ntargets, const int64_t *targets,
                         double *ax, double *ay, double *az, uint32_t *nbr, double *min_gap)
{
    double c[6];
    for (int k = 0; k < 6; ++k) c[k] = (double)poly_f[k];
    const double eps = (double)eps_f;
    const double rm2 = (double)r_max * (double)r_max;
    const int64_t nt = targets ? ntargets : n;
    uint64_t total = 0;
    double gap = 1e300;
#pragma omp parallel for schedule(dynamic, 8) reduction(+ : total) reduction(min : gap)
    for (int64_t t = 0; t < nt; ++t) {
        const int64_t i = targets ? targets[t] : t;
        const double xi = x[i], yi = y[i], zi = z[i];
        double sx = 0.0, sy = 0.0, sz = 0.0;
        uint32_t cnt = 0;
        for (int64_t j = 0; j < n; ++j) {
            if (j == i) continue;
            double dx = min_image((double)x[j] - xi, L);
            double dy = min_image((double)y[j] - yi, L);
            double dz = min_image((double)z[j] - zi, L);
            double s = dx * dx + dy * dy + dz * dz;
            double gp = fabs(s - rm2) / rm2;
            if (gp < gap) gap = gp;
            if (s < rm2) {
                double f = (m ? (double)m[j] : 1.0) * (pow(s + eps, -1.5) - poly5(s, c));
                sx += f * dx;
                sy += f * dy;
                sz += f * dz;
                ++cnt;
            }
        }
        ax[t] = sx;
        ay[t] = sy;
        az[t] = sz;
        if (nbr) nbr[t] = cnt;
        total += cnt;
    }
    if (min_gap) *min_gap = gap;
    return total;
}

/* Exact cell coordinate floor(x*nc/L) (reading S12): the product of a float32 and a small
 * integer is exact in double, and L is a power of two in every config. */
static inline int cell_coord(float x, int nc, double L)
{
    int c = (int)floor((double)x * (double)nc / L);
    if (c < 0) c = 0;
    if (c > nc - 1) c = nc - 1;
    return c;
}

/*
 * Chaining mesh (readings S12, S13): cid = cx + nc*(cy + nc*cz);
 * count = histogram; cell_start = exclusive prefix sum, cell_start[nc^3] = n.
 */
void oracle_mesh(int64_t n, const float *x, const float *y, const float *z, double L, int nc,
                 uint32_t *cid, uint32_t *count, uint32_t *cell_start)
{
    const int64_t ncell = (int64_t)nc * nc * nc;
    memset(count, 0, sizeof(uint32_t) * (size_t)ncell);
    for (int64_t i = 0; i < n; ++i) {
        int cx = cell_coord(x[i], nc, L), cy = cell_coord(y[i], nc, L),
            cz = cell_coord(z[i], nc, L);
        uint32_t c = (uint32_t)(cx + nc * (cy + nc * cz));
        cid[i] = c;
        count[c]++;
    }
    uint32_t run = 0;
    for (int64_t c = 0; c < ncell; ++c) {
        cell_start[c] = run;
        run += count[c];
    }
    cell_start[ncell] = run;
}

/*
 * Independent cell-list evaluation: Hockney & Eastwood linked list (head/next), not a
 * counting sort.  Same outputs as the brute force (targets == NULL -> all particles, else the
 * ntargets listed ones, outputs indexed by position in the list); with want_force == 0 only
 * the neighbour counts are produced.  seconds (may be NULL) receives {list build, evaluation}
 * wall times, for bench.py's cpu_baseline.  Requires nc >= 3 and L/nc >= r_max.  n_eval (may be NULL)
 * receives the number of candidate (evaluated) ordered pairs sum_c n_c * sum_{27} n_c'
 * minus the n self pairs.
 */
uint64_t oracle_sr_celllist(int64_t n, const float *x, const float *y, const float *z,
                            const float *m, double L, int nc, float r_max, float eps_f,
                            const float poly_f[6], int want_force, int64_t ntargets,
                            const int64_t *targets, double *ax, double *ay, double *az,
                            uint32_t *nbr, uint64_t *n_eval, double *seconds)
{
    double c[6];
    for (int k = 0; k < 6; ++k) c[k] = (double)poly_f[k];
    const double eps = (double)eps_f;
    const double rm2 = (double)r_max * (double)r_max;
    const int64_t ncell = (int64_t)nc * nc * nc;
    int64_t *head = (int64_t *)malloc(sizeof(int64_t) * (size_t)ncell);
    int64_t *next = (int64_t *)malloc(sizeof(int64_t) * (size_t)(n > 0 ? n : 1));
    int32_t *pc = (int32_t *)malloc(sizeof(int32_t) * 3 * (size_t)(n > 0 ? n : 1));
    double t0 = 0.0, t1 = 0.0, t2 = 0.0;
#ifdef _OPENMP
    t0 = omp_get_wtime();
#endif
    for (int64_t q = 0; q < ncell; ++q) head[q] = -1;
    for (int64_t i = n - 1; i >= 0; --i) {
        int cx = cell_coord(x[i], nc, L), cy = cell_coord(y[i], nc, L),
            cz = cell_coord(z[i], nc, L);
        pc[3 * i] = cx;
        pc[3 * i + 1] = cy;
        pc[3 * i + 2] = cz;
        int64_t q = cx + (int64_t)nc * (cy + (int64_t)nc * cz);
        next[i] = head[q];
        head[q] = i;
    }
    uint64_t total = 0, evals = 0;
    const int64_t nt = targets ? ntargets : n;
#ifdef _OPENMP
    t1 = omp_get_wtime();
#endif
#pragma omp parallel for schedule(dynamic, 64) reduction(+ : total, evals)
    for (int64_t t = 0; t < nt; ++t) {
        const int64_t i = targets ? targets[t] : t;
        const double xi = x[i], yi = y[i], zi = z[i];
        double sx = 0.0, sy = 0.0, sz = 0.0;
        uint32_t cnt = 0;
        for (int oz = -1; oz <= 1; ++oz)
            for (int oy = -1; oy <= 1; ++oy)
                for (int ox = -1; ox <= 1; ++ox) {
                    int qx = (pc[3 * i] + ox + nc) % nc, qy = (pc[3 * i + 1] + oy + nc) % nc,
                        qz = (pc[3 * i + 2] + oz + nc) % nc;
                    int64_t q = qx + (int64_t)nc * (qy + (int64_t)nc * qz);
                    for (int64_t j = head[q]; j >= 0; j = next[j]) {
                        if (j == i) continue;
                        ++evals;
                        double dx = min_image((double)x[j] - xi, L);
                        double dy = min_image((double)y[j] - yi, L);
                        double dz = min_image((double)z[j] - zi, L);
                        double s = dx * dx + dy * dy + dz * dz;
                        if (s < rm2) {
                            ++cnt;
                            if (want_force) {
                                double f = (m ? (double)m[j] : 1.0) *
                                           (pow(s + eps, -1.5) - poly5(s, c));
                                sx += f * dx;
                                sy += f * dy;
                                sz += f * dz;
                            }
                        }
                    }
                }
        if (want_force) {
            ax[t] = sx;
            ay[t] = sy;
            az[t] = sz;
        }
        if (nbr) nbr[t] = cnt;
        total += cnt;
    }
#ifdef _OPENMP
    t2 = omp_get_wtime();
#endif
    if (seconds) {
        seconds[0] = t1 - t0;
        seconds[1] = t2 - t1;
    }
    free(head);
    free(next);
    free(pc);
    if (n_eval) *n_eval = evals;
    return total;
}

/* Kick map: v <- v + dt * a  (double result from float32 v and double a). */
void oracle_kick(int64_t n, const float *v, const double *a, float dt, double *v_out)
{
    for (int64_t i = 0; i < n; ++i) v_out[i] = (double)v[i] + (double)dt * a[i];
}

/* Stream map, with the wrap rule of reading S16:
 * x <- x + dt*v;  x <- x - L*floor(x/L).  Result in double, in [0, L). */
void oracle_drift(int64_t n, const float *x, const float *v, float dt, double L, double *x_out)
{
    for (int64_t i = 0; i < n; ++i) {
        double p = (double)x[i] + (double)dt * (double)v[i];
        p -= L * floor(p / L);
        if (p >= L) p = 0.0;
        x_out[i] = p;
    }
}
