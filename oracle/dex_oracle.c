/*
 * dex_oracle.c -- CPU ORACLE for the long-characteristics formal solution of
 * arxiv/paper_2511_08498 ("A Simple Ray Acceleration Structure for Non-LTE
 * Radiative Transfer").
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may build, load or call it.
 * It shares no code with the CUDA library (paper_2511_08498_b200/csrc): no headers,
 * no helpers, no tables.  It is deliberately plain and slow: fp64 intensities, one ray
 * at a time, no blocking / fusion / reordering beyond what the cited passage states.
 *
 * Contents (each function cites the passage it follows; PAPER.md = /root/reference/PAPER.md,
 * T-/V-rules = SURVEY.md section 8(c), restated in DESIGN.md):
 *   orc_segment            eq. 3 with constant eta, chi in a cell
 *   orc_voigt_H            HUM1WEI24 Voigt function
 *   orc_line_terms         eqs. 10-20 line emissivity / opacity
 *   orc_plain_march        (A) AW87 DDA through every level-0 voxel
 *   orc_hdda_march         (B) HDDA over the brick/level structure (Algorithm 1)
 *   orc_mean_intensity     J = sum_k w_k I_k
 *
 * Parity pins (tests/test_oracle_*.py): homogeneous slab closed form, Table 1 "Average"
 * column, transparency of chi=0 voxels, thin limit, HDDA == plain DDA invariants, brute-force
 * slab intersection on tiny grids, scipy.special.wofz for the Voigt function.
 * Unpinned (geometry/data not in the paper text): Table 1 "True" column, Tables 2-3.
 *
 * Build: gcc -O2 -std=c11 -ffp-contract=off -fno-fast-math -fopenmp -shared -fPIC
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#include <complex.h>
#undef I /* the name I is used for intensities below; the imaginary unit is _Complex_I */
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_MAX_LINES 4 /* max overlapping lines is a compile-time 4 */
#define ORC_MAX_W 64

/* ------------------------------------------------------------------------------------ */
/* eq. 3 with piecewise-constant eta, chi                         */
/*   I_out = I_in e^{-tau} + S (1 - e^{-tau}),  tau = chi * (h ds),  S = eta / chi        */
/* written with E(tau) = (1 - e^{-tau}) / tau so that chi = 0 is the limit                */
/*   I_out = I_in + eta * (h ds)      (E(0) = 1)                          */
/* ------------------------------------------------------------------------------------ */
double orc_segment(double I_in, double eta, double chi, double hds)
{
    double tau = chi * hds;
    double E = (tau > 0.0) ? (-expm1(-tau) / tau) : 1.0;
    return I_in * exp(-tau) + eta * hds * E;
}

/* ------------------------------------------------------------------------------------ */
/* Voigt function H(a,x) = Re w(x + i a), "HUM1WEI24" of Schreier (2018):  */
/*   |x| + a >= 15 : Humlicek (1982) region I,  w = (i/sqrt(pi)) z / (z^2 - 1/2)          */
/*   otherwise     : Weideman (1994) N = 24 rational expansion                            */
/*       L = 2^{-1/4} N^{1/2},  Z = (L + i z)/(L - i z),                                  */
/*       w = 2 p(Z)/(L - i z)^2 + (1/sqrt(pi))/(L - i z),  p(Z) = sum_{n=1}^{N} c_n Z^{n-1}*/
/*   c_n are the Fourier coefficients of f(t) = e^{-t^2}(L^2 + t^2) under t = L tan(th/2):*/
/*       c_n = (1/(4N)) sum_{k=-(2N-1)}^{2N-1} f(t_k) cos(n th_k),  th_k = k pi/(2N).     */
/* The coefficients are not printed in the paper; they are computed here by the direct    */
/* cosine sum above (no table copied from anywhere).                                      */
/* ------------------------------------------------------------------------------------ */
#define WEI_N 24
static double wei_c[WEI_N + 1];
static double wei_L;
static int wei_ready = 0;

static void wei_init(void)
{
    if (wei_ready) return;
    const int N = WEI_N, M = 2 * N;
    const double L = sqrt((double)N / sqrt(2.0));
    for (int n = 1; n <= N; ++n) {
        double s = 0.0;
        for (int k = -(M - 1); k <= M - 1; ++k) {
            double th = (double)k * M_PI / (double)M;
            double t = L * tan(0.5 * th);
            double f = exp(-t * t) * (L * L + t * t);
            s += f * cos((double)n * th);
        }
        wei_c[n] = s / (2.0 * (double)M);
    }
    wei_L = L;
    wei_ready = 1;
}

void orc_init(void) { wei_init(); }

double orc_voigt_H(double a, double x)
{
    if (!wei_ready) wei_init();
    double complex z = x + _Complex_I * a;
    if (fabs(x) + a >= 15.0) {
        double complex w = (_Complex_I / sqrt(M_PI)) * z / (z * z - 0.5);
        return creal(w);
    }
    double complex lmiz = wei_L - _Complex_I * z;
    double complex Z = (wei_L + _Complex_I * z) / lmiz;
    double complex p = wei_c[WEI_N];
    for (int n = WEI_N - 1; n >= 1; --n) p = p * Z + wei_c[n];
    double complex w = 2.0 * p / (lmiz * lmiz) + (1.0 / sqrt(M_PI)) / lmiz;
    return creal(w);
}

void orc_voigt_H_array(const double* a, const double* x, double* out, int64_t n)
{
    wei_init();
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) out[i] = orc_voigt_H(a[i], x[i]);
}

/* ------------------------------------------------------------------------------------ */
/* Line emissivity / opacity of one line at one wavelength:            */
/*   eta_l = eta*_l(lambda) phi_l,  chi_l = chi*_l(lambda) phi_l             (eqs. 15-16)  */
/*   eta*(lambda) = (lambda0/lambda) eta*(lambda0), chi* likewise            (eqs. 18-19)  */
/*   a(lambda) = (lambda/lambda0)^2 a(lambda0)                               (eq. 20)      */
/*   phi_l(lambda, w) = varphi_l(lambda + (v.w/c) lambda0)                   (eq. 14)      */
/*   varphi = H(a, x) / (sqrt(pi) dlamD),  x = (lambda' - lambda0)/dlamD  (standard Voigt  */
/*   normalisation; the paper does not print it -- DESIGN.md reading R-phi)                */
/* vproj = v . omega-hat in the units of c_light.                                          */
/* ------------------------------------------------------------------------------------ */
void orc_line_terms(double lam, double lam0, double eta_star0, double chi_star0, double a0,
                    double inv_dlamD, double vproj, double c_light, double* eta_l, double* chi_l)
{
    double x = ((lam - lam0) + (vproj / c_light) * lam0) * inv_dlamD;
    double r = lam / lam0;
    double a = r * r * a0;
    double phi = orc_voigt_H(a, x) * inv_dlamD / sqrt(M_PI);
    double s = lam0 / lam;
    *eta_l = s * eta_star0 * phi;
    *chi_l = s * chi_star0 * phi;
}

/* ------------------------------------------------------------------------------------ */
/* Field description handed over by oracle.py.  Level m arrays are DENSE over the whole   */
/* level-m grid: cell (cx,cy,cz) -> ((cz*Ny_m + cy)*Nx_m + cx), N_m = N >> m.            */
/* ------------------------------------------------------------------------------------ */
typedef struct {
    int variant;                 /* 0 ISO, 1 VELINTERP, 2 CAV, 3 CLASSIC */
    int n_lambda;
    int W;                       /* wavelengths per batch (8) */
    int n_levels;                /* number of levels present in the per-level arrays */
    const float* const* eta;     /* [level] -> [cells][n_lambda]; ISO: eta, CAV/CLASSIC: eta_bg */
    const float* const* chi;
    const float* lam;            /* [n_lambda] */
    int n_lines;
    const float* lambda0;        /* [n_lines] */
    const float* const* eta_star;/* [level] -> [n_lines][cells] */
    const float* const* chi_star;
    const float* const* a0;
    const float* const* inv_dlamD;
    const float* const* vbar;    /* [level] -> [cells][ndim] box-filtered velocity */
    const int8_t* active_lines;  /* [n_batch][ORC_MAX_LINES], -1 padded */
    double c_light;
    int n_vbins;                 /* VELINTERP */
    const float* const* vtab;    /* [level] -> [cells][n_vbins][n_lambda][2] (eta, chi) */
    const float* const* vmax;    /* [level] -> [cells] half-width of the velocity grid */
} orc_fields;

typedef struct {
    int ndim;
    int dims[3];
    int brick;
    double h;                    /* physical side of a level-0 voxel */
    /* Distance-dependent MIP cap, the long-characteristics analogue of DexRT's per-cascade maximum MIP level
     * [0,0,1,2,3,4] with interval ends 1.5 * 4^i voxels (T8): a cell
     * entered at distance t from the probe is formed at level min(brick level, #{i : t >= cap_t[i]}).
     * n_caps = 0: no cap. */
    int n_caps;
    float cap_t[8];              /* ascending thresholds, index units */
    /* 2.5D rays (in-plane angular samples "augmented with a 4 sample Gauss-Radau quadrature for
     * different inclinations in y", y homogeneous and without velocity components): direction k
     * makes the angle theta_k with the homogeneous axis, sin_incl[k] = sin(theta_k).  The traversal is the in-plane
     * one; every path length is divided by sin(theta) and the in-plane direction that projects the velocity is
     * multiplied by it.  NULL: rays lie in the plane.  2D grids only. */
    const float* sin_incl;       /* [n_dirs] or NULL */
    /* Finite radiance interval (DexRT traces HDDA(t1, t2) per cascade, Algorithm 1 l.9 and PAPER.md:347; SURVEY.md
     * 8(f)-4; T10): only the part of the ray with t in [t_begin, t_end] (index units, from the probe)
     * contributes.  The traversal itself is unchanged and starts at the probe, so the cells and plane times are
     * those of the full ray; each visit [t, t_h] is clipped to the interval.  t_end <= 0: to the boundary. */
    float t_begin, t_end;
} orc_grid;

/* T10: clip the visit [t, th] to the interval; returns the clipped length (<= 0: nothing to emit) */
static inline float clip_visit(const orc_grid* g, float t, float th)
{
    if (g->t_end <= 0.0f) return th - t;
    return fminf(th, g->t_end) - fmaxf(t, g->t_begin);
}

static inline int64_t cell_index(const orc_grid* g, int m, const int* cc)
{
    int64_t nx = g->dims[0] >> m, ny = g->dims[1] >> m;
    int64_t cz = (g->ndim == 3) ? cc[2] : 0;
    return (cz * ny + cc[1]) * nx + cc[0];
}

/* VELINTERP lookup (reading R-vel): linear interpolation of the
 * n-bin table on the uniform grid [-V, V] at projected velocity v, clamped to the grid.  */
static void velinterp_lookup(const float* tab, int n_vbins, int n_lambda, int lam0, int W,
                             double V, double v, double* eta, double* chi)
{
    int i0 = 0;
    double w = 0.0;
    if (V > 0.0 && n_vbins > 1) {
        double f = (v + V) / (2.0 * V) * (double)(n_vbins - 1);
        if (f < 0.0) f = 0.0;
        if (f > (double)(n_vbins - 1)) f = (double)(n_vbins - 1);
        i0 = (int)floor(f);
        if (i0 > n_vbins - 2) i0 = n_vbins - 2;
        w = f - (double)i0;
    }
    int i1 = (n_vbins > 1) ? i0 + 1 : i0;
    for (int j = 0; j < W; ++j) {
        const float* p0 = tab + ((int64_t)i0 * n_lambda + (lam0 + j)) * 2;
        const float* p1 = tab + ((int64_t)i1 * n_lambda + (lam0 + j)) * 2;
        eta[j] = (1.0 - w) * (double)p0[0] + w * (double)p1[0];
        chi[j] = (1.0 - w) * (double)p0[1] + w * (double)p1[1];
    }
}

/* eta, chi of one cell for the W wavelengths of batch b, seen along propagation direction w. */
static void provider(const orc_grid* g, const orc_fields* F, int m, int64_t cell, int b,
                     const double* omega, double* eta, double* chi)
{
    const int W = F->W, nl = F->n_lambda, l0 = b * W;
    if (F->variant == 0) {
        for (int j = 0; j < W; ++j) {
            eta[j] = (double)F->eta[m][cell * nl + l0 + j];
            chi[j] = (double)F->chi[m][cell * nl + l0 + j];
        }
        return;
    }
    int64_t ncell = 1;
    for (int a = 0; a < g->ndim; ++a) ncell *= (g->dims[a] >> m);
    double vproj = 0.0;
    for (int a = 0; a < g->ndim; ++a) vproj += (double)F->vbar[m][cell * g->ndim + a] * omega[a];
    if (F->variant == 1) {
        const float* tab = F->vtab[m] + cell * (int64_t)F->n_vbins * nl * 2;
        velinterp_lookup(tab, F->n_vbins, nl, l0, W, (double)F->vmax[m][cell], vproj, eta, chi);
        return;
    }
    /* CAV / CLASSIC: eqs. 10-11 */
    for (int j = 0; j < W; ++j) {
        double e = (double)F->eta[m][cell * nl + l0 + j];
        double c = (double)F->chi[m][cell * nl + l0 + j];
        double lam = (double)F->lam[l0 + j];
        for (int q = 0; q < ORC_MAX_LINES; ++q) {
            int l = F->active_lines[b * ORC_MAX_LINES + q];
            if (l < 0) continue;
            double el, cl;
            orc_line_terms(lam, (double)F->lambda0[l], (double)F->eta_star[m][l * ncell + cell],
                           (double)F->chi_star[m][l * ncell + cell], (double)F->a0[m][l * ncell + cell],
                           (double)F->inv_dlamD[m][l * ncell + cell], vproj, F->c_light, &el, &cl);
            e += el;
            c += cl;
        }
        eta[j] = e;
        chi[j] = c;
    }
}

/* T2: time of the grid plane with integer coordinate k on axis a is a pure
 * function of (ray, a, k): one fused multiply-add, no accumulation.                         */
static inline float tplane(int k, float inv, float off) { return fmaf((float)k, inv, off); }

typedef struct {
    int level;
    int cc[3];     /* cell coordinate at that level (level-0 coordinate >> level) */
    float ds;      /* t_h - t in index units, fp32 */
} seg_t;

static inline uint64_t pack_record(const seg_t* s)
{
    /* T7: canonical, storage-independent visit record */
    return ((uint64_t)(uint8_t)s->level << 56) | ((uint64_t)(uint32_t)s->cc[2] << 36) |
           ((uint64_t)(uint32_t)s->cc[1] << 18) | (uint64_t)(uint32_t)s->cc[0];
}

/* ray set-up, T1/T2: trace from the probe outward, o = probe, d = -omega */
typedef struct { float o[3], d[3], inv[3], off[3]; int nz[3]; } ray_t;

static int ray_setup(const orc_grid* g, const float* probe, const float* omega, ray_t* r, int* x0)
{
    int any = 0;
    for (int a = 0; a < 3; ++a) { r->o[a] = 0.f; r->d[a] = 0.f; r->inv[a] = 0.f; r->off[a] = 0.f; r->nz[a] = 0; x0[a] = 0; }
    for (int a = 0; a < g->ndim; ++a) {
        r->o[a] = probe[a];
        r->d[a] = -omega[a];
        if (r->d[a] != 0.0f) {
            r->nz[a] = 1;
            any = 1;
            r->inv[a] = 1.0f / r->d[a];
            r->off[a] = -r->o[a] * r->inv[a];
        }
        x0[a] = (int)floorf(r->o[a]);          /* T6 */
        if (x0[a] < 0 || x0[a] >= g->dims[a]) return 0;
    }
    return any;
}

/* ------------------------------------------------------------------------------------ */
/* (A) plain march: AW87 DDA through every level-0 voxel ("essentially       */
/* matching that of AW87"), T-rules with size == 1 everywhere.  Returns the number of     */
/* segments written (all voxels crossed with t_h > t, empty ones included).               */
/* ------------------------------------------------------------------------------------ */
static int plain_dda(const orc_grid* g, const float* probe, const float* omega, seg_t* segs, int max_segs)
{
    ray_t r;
    int x[3];
    if (!ray_setup(g, probe, omega, &r, x)) return 0;
    float t = 0.0f;
    int n = 0;
    for (;;) {
        int s = -1;
        float th = INFINITY;
        for (int a = 0; a < g->ndim; ++a) {
            if (!r.nz[a]) continue;
            int kp = (r.d[a] > 0.0f) ? x[a] + 1 : x[a];     /* T3 with size 1 */
            float tn = tplane(kp, r.inv[a], r.off[a]);
            if (s < 0 || tn < th) { th = tn; s = a; }         /* T4: lowest-index axis attaining the min */
        }
        if (th > t && clip_visit(g, t, th) > 0.0f) {
            if (n >= max_segs) return -1;
            segs[n].level = 0;
            segs[n].cc[0] = x[0]; segs[n].cc[1] = x[1]; segs[n].cc[2] = x[2];
            segs[n].ds = clip_visit(g, t, th);
            ++n;
        }
        if (th > t) t = th;
        if (g->t_end > 0.0f && t >= g->t_end) break;           /* T10: the interval ends inside the grid */
        x[s] += (r.d[s] > 0.0f) ? 1 : -1;                      /* T5 with size 1 */
        if (x[s] < 0 || x[s] >= g->dims[s]) break;
    }
    return n;
}

/* ------------------------------------------------------------------------------------ */
/* (B) HDDA (Algorithm 1) under the T-rules.  `level` is the brick      */
/* table of one batch: -1 empty, else the MIP level of the whole brick.    */
/* Emits only non-empty cells with t_h > t (T4).                                          */
/* ------------------------------------------------------------------------------------ */
static inline int brick_index(const orc_grid* g, const int* x)
{
    int B = g->brick;
    int nbx = g->dims[0] / B, nby = g->dims[1] / B;
    int bz = (g->ndim == 3) ? x[2] / B : 0;
    return (bz * nby + x[1] / B) * nbx + x[0] / B;
}

static int hdda(const orc_grid* g, const int8_t* level, const float* probe, const float* omega,
                seg_t* segs, int max_segs)
{
    ray_t r;
    int x[3];   /* level-0 voxel containing the ray ("coord" of Algorithm 1 before FloorToStep) */
    if (!ray_setup(g, probe, omega, &r, x)) return 0;
    float t = 0.0f;
    int n = 0;
    for (;;) {
        int m = level[brick_index(g, x)];                       /* MipLevel(coord), Alg. 1 l.6-8 */
        if (m > 0 && g->n_caps > 0) {                            /* T8: near field at fine resolution */
            int cap = 0;
            for (int i = 0; i < g->n_caps; ++i) cap += (t >= g->cap_t[i]) ? 1 : 0;
            if (cap < m) m = cap;
        }
        int size = (m < 0) ? g->brick : (1 << m);                /* T3: empty brick skipped whole */
        int c[3], kp[3];
        int s = -1;
        float th = INFINITY;
        for (int a = 0; a < g->ndim; ++a) {
            c[a] = x[a] & ~(size - 1);                           /* FloorToStep, Alg. 1 l.1-5 */
            if (!r.nz[a]) continue;
            kp[a] = (r.d[a] > 0.0f) ? c[a] + size : c[a];        /* NextPlaneHit */
            float tn = tplane(kp[a], r.inv[a], r.off[a]);
            if (s < 0 || tn < th) { th = tn; s = a; }
        }
        if (m >= 0 && th > t && clip_visit(g, t, th) > 0.0f) {   /* "Integrate RTE over [t, t_h]" l.25-26 */
            if (n >= max_segs) return -1;
            segs[n].level = m;
            segs[n].cc[0] = c[0] >> m; segs[n].cc[1] = c[1] >> m; segs[n].cc[2] = (g->ndim == 3) ? (c[2] >> m) : 0;
            segs[n].ds = clip_visit(g, t, th);
            ++n;
        }
        if (th > t) t = th;
        if (g->t_end > 0.0f && t >= g->t_end) break;             /* T10: "while t < t2", Alg. 1 l.22 */
        /* T5: cross plane (s, kp[s]); the other axes take the level-0 coordinate the plain DDA
         * would hold at this event: plane (a,k) counts as crossed iff tplane < t_h, or == t_h
         * and a < s (lower-index axes go first in ties).                                      */
        int xs = (r.d[s] > 0.0f) ? kp[s] : kp[s] - 1;
        if (xs < 0 || xs >= g->dims[s]) break;
        if (size > 1) {
            for (int a = 0; a < g->ndim; ++a) {
                if (a == s || !r.nz[a]) continue;
                int lo = c[a], hi = c[a] + size - 1;
                if (r.d[a] > 0.0f) {
                    int xa = lo;
                    for (int k = lo + 1; k <= hi; ++k) {
                        float tp = tplane(k, r.inv[a], r.off[a]);
                        if (tp < th || (tp == th && a < s)) xa = k; else break;
                    }
                    x[a] = xa;
                } else {
                    int xa = hi;
                    for (int k = hi - 1; k >= lo; --k) {
                        float tp = tplane(k + 1, r.inv[a], r.off[a]);
                        if (tp < th || (tp == th && a < s)) xa = k; else break;
                    }
                    x[a] = xa;
                }
            }
        }
        x[s] = xs;
    }
    return n;
}

/* Apply eq. 3 from the boundary to the probe over a collected segment list (north_star
 * recurrence I_out = I_in e^{-chi ds} + S (1 - e^{-chi ds})), for the W wavelengths of batch b. */
static void integrate_list(const orc_grid* g, const orc_fields* F, const seg_t* segs, int n, int b,
                           const double* omega, double sin_incl, const float* i0_dir, double* I_out)
{
    const int W = F->W;
    double I[ORC_MAX_W], eta[ORC_MAX_W], chi[ORC_MAX_W];
    for (int j = 0; j < W; ++j) I[j] = i0_dir ? (double)i0_dir[b * W + j] : 0.0;
    for (int i = n - 1; i >= 0; --i) {
        int64_t cell = cell_index(g, segs[i].level, segs[i].cc);
        provider(g, F, segs[i].level, cell, b, omega, eta, chi);
        double hds = g->h * (double)segs[i].ds / sin_incl;        /* 3D path length of the in-plane segment */
        for (int j = 0; j < W; ++j) I[j] = orc_segment(I[j], eta[j], chi[j], hds);
    }
    for (int j = 0; j < W; ++j) I_out[b * W + j] = I[j];
}

/* capture buffers (validation): per ray `cap_stride` records */
typedef struct {
    int64_t* counts;    /* [n_rays] */
    uint64_t* records;  /* [n_rays][cap_stride] */
    float* ds;          /* [n_rays][cap_stride] */
    int cap_stride;
    int batch;          /* which batch's traversal to capture (HDDA) */
} orc_capture;

static void capture_store(orc_capture* cap, int64_t ray, const seg_t* segs, int n)
{
    cap->counts[ray] = n;
    int m = n < cap->cap_stride ? n : cap->cap_stride;
    for (int i = 0; i < m; ++i) {
        cap->records[ray * cap->cap_stride + i] = pack_record(&segs[i]);
        cap->ds[ray * cap->cap_stride + i] = segs[i].ds;
    }
}

static int max_segments(const orc_grid* g)
{
    int n = 8;
    for (int a = 0; a < g->ndim; ++a) n += g->dims[a] + 2;
    return n;
}

/* I[probe][dir][lambda] (double).  Returns emitted-segment count summed over rays and batches,
 * or -1 on error.  In the plain march a "segment" is counted only where chi or eta can be
 * nonzero is NOT known to it, so it counts every crossed voxel (per batch).                  */
int64_t orc_plain_march(const orc_grid* g, const orc_fields* F, int64_t n_probes, const float* probe_pos,
                        int n_dirs, const float* dirs, const float* i0, double* I, orc_capture* cap,
                        int n_threads)
{
    wei_init();
    if (F->W > ORC_MAX_W || F->n_lambda % F->W) return -1;
    const int nb = F->n_lambda / F->W, ms = max_segments(g);
    int64_t total = 0;
    int err = 0;
#ifdef _OPENMP
    if (n_threads > 0) omp_set_num_threads(n_threads);
#endif
#pragma omp parallel reduction(+ : total)
    {
        seg_t* segs = (seg_t*)malloc(sizeof(seg_t) * (size_t)ms);
#pragma omp for schedule(dynamic, 4)
        for (int64_t p = 0; p < n_probes; ++p) {
            for (int k = 0; k < n_dirs; ++k) {
                const float* om = dirs + (int64_t)k * g->ndim;
                double omega[3] = {0, 0, 0};
                const double si = (g->sin_incl && g->ndim == 2) ? (double)g->sin_incl[k] : 1.0;
                for (int a = 0; a < g->ndim; ++a) omega[a] = (double)om[a] * si;   /* in-plane part of the 3D direction */
                int n = plain_dda(g, probe_pos + p * g->ndim, om, segs, ms);
                if (n < 0) { err = 1; n = 0; }
                int64_t ray = p * n_dirs + k;
                if (cap) capture_store(cap, ray, segs, n);
                for (int b = 0; b < nb; ++b)
                    integrate_list(g, F, segs, n, b, omega, si, i0 ? i0 + (int64_t)k * F->n_lambda : NULL,
                                   I + ray * F->n_lambda);
                total += (int64_t)n * nb;
            }
        }
        free(segs);
    }
    return err ? -1 : total;
}

int64_t orc_hdda_march(const orc_grid* g, const orc_fields* F, const int8_t* levels /*[n_batch][n_bricks]*/,
                       int64_t n_probes, const float* probe_pos, int n_dirs, const float* dirs,
                       const float* i0, double* I, orc_capture* cap, int n_threads)
{
    wei_init();
    if (F->W > ORC_MAX_W || F->n_lambda % F->W) return -1;
    const int nb = F->n_lambda / F->W, ms = max_segments(g);
    int64_t n_bricks = 1;
    for (int a = 0; a < g->ndim; ++a) n_bricks *= g->dims[a] / g->brick;
    int64_t total = 0;
    int err = 0;
#ifdef _OPENMP
    if (n_threads > 0) omp_set_num_threads(n_threads);
#endif
#pragma omp parallel reduction(+ : total)
    {
        seg_t* segs = (seg_t*)malloc(sizeof(seg_t) * (size_t)ms);
#pragma omp for schedule(dynamic, 4)
        for (int64_t p = 0; p < n_probes; ++p) {
            for (int k = 0; k < n_dirs; ++k) {
                const float* om = dirs + (int64_t)k * g->ndim;
                double omega[3] = {0, 0, 0};
                const double si = (g->sin_incl && g->ndim == 2) ? (double)g->sin_incl[k] : 1.0;
                for (int a = 0; a < g->ndim; ++a) omega[a] = (double)om[a] * si;   /* in-plane part of the 3D direction */
                int64_t ray = p * n_dirs + k;
                for (int b = 0; b < nb; ++b) {
                    int n = hdda(g, levels + (int64_t)b * n_bricks, probe_pos + p * g->ndim, om, segs, ms);
                    if (n < 0) { err = 1; n = 0; }
                    if (cap && cap->batch == b) capture_store(cap, ray, segs, n);
                    integrate_list(g, F, segs, n, b, omega, si, i0 ? i0 + (int64_t)k * F->n_lambda : NULL,
                                   I + ray * F->n_lambda);
                    total += n;
                }
            }
        }
        free(segs);
    }
    return err ? -1 : total;
}

/* J(p, lambda) = sum_k w_k I(p, k, lambda)   (directions and weights are inputs) */
void orc_mean_intensity(int64_t n_probes, int n_dirs, int n_lambda, const float* weights,
                        const double* I, double* J)
{
    for (int64_t p = 0; p < n_probes; ++p)
        for (int j = 0; j < n_lambda; ++j) {
            double s = 0.0;
            for (int k = 0; k < n_dirs; ++k) s += (double)weights[k] * I[(p * n_dirs + k) * n_lambda + j];
            J[p * n_lambda + j] = s;
        }
}

int orc_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
