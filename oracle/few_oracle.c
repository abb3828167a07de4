/* few_oracle.c -- CPU ORACLE for the FastEMRIWaveforms interpolated mode summation.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may build, load or call it.  It shares no code, header, table or
 * helper with the CUDA path under paper_2104_04582_b200/csrc/ and neither includes the other.
 *
 * It is deliberately plain and slow: a Thomas solve per spline, a comparison sort per time step, a direct
 * loop over modes per sample, phases in x87 extended precision (64-bit mantissa).  Every function cites the
 * passage of /root/reference/PAPER.md (arXiv 2104.04582) it follows; where the paper is silent the reading
 * is the one listed in DESIGN.md ("Readings", R1..R19).
 *
 * Pins (tests/test_oracle_pins.py, all `-m "not gpu"`):
 *   oracle_spline_fit / _ext : P1 cubic reproduction, P2 dense LU of the un-eliminated system + continuity,
 *                              P3 SciPy not-a-knot CubicSpline, P7 mpmath brute force.
 *   oracle_ylm               : P6 l=2 closed forms, orthonormality under quadrature, poles, m -> -m symmetry.
 *   oracle_select_modes      : P8 brute-force prefix enumeration on tiny inputs + invariants.
 *   oracle_sum_waveform      : P4 closed form, P5 m -> -m fold vs explicit negative-m list, P7 mpmath brute
 *                              force (config 0), P9 real-linearity, P10 time translation / batch independence.
 *   oracle_frame / _apply    : P12 wave-frame geometry rebuilt from Eq. (4)-(7) with cross products, spin-2 tensor
 *                              projection, norm preservation, invariance under a common rotation about z.
 *   oracle_inner             : P13 Parseval against the frequency-domain form of Eq. (16) (numpy FFT), overlap(a,a)=1.
 *   oracle_sum_direct        : P14 closed form, mpmath brute force, agreement with the interpolated sum on inputs
 *                              that are exactly cubic per segment.
 *   oracle_sum_waveform_kerr : P15 equals oracle_sum_waveform for k = 0 / two phases, single-mode closed form with k,
 *                              (-1)^(l+k) fold vs the explicit (l,-m,-k,-n) list, mpmath brute force with three phases.
 * No function here is "parity unpinned".
 *
 * Build: gcc -O2 -fopenmp -ffp-contract=off -shared -fPIC few_oracle.c -o libfew_oracle.so -lm
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef long double ext; /* x86-64: 80-bit, 64-bit mantissa (reading R13) */

int oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void oracle_set_threads(int n)
{
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

/* ------------------------------------------------------------------------------------------------
 * O1 -- not-a-knot cubic spline on a shared sparse grid (sec. III C: "The specific spline
 * implemented is the 'not-a-knot' spline ... tridiagonal banded matrix representation ... all arrays to be
 * interpolated exist on the same sparse time grid").
 *
 * Unknowns s_i = S'(t_i).  h_i = t_{i+1}-t_i, delta_i = (y_{i+1}-y_i)/h_i.
 *   interior  i=1..n-2 :  h_i s_{i-1} + 2(h_{i-1}+h_i) s_i + h_{i-1} s_{i+1} = 3 (h_i delta_{i-1} + h_{i-1} delta_i)
 *   first row          :  h_1 s_0 + (h_0+h_1) s_1 = [ (3h_0+2h_1) h_1 delta_0 + h_0^2 delta_1 ] / (h_0+h_1)
 *   last row           :  (h_{n-2}+h_{n-3}) s_{n-2} + h_{n-3} s_{n-1}
 *                             = [ h_{n-2}^2 delta_{n-3} + (2h_{n-3}+3h_{n-2}) h_{n-3} delta_{n-2} ] / (h_{n-3}+h_{n-2})
 * (third-derivative continuity at t_1 and t_{n-2} with the far unknown eliminated, so the system stays
 * tridiagonal).  Thomas elimination, no pivoting.  Per segment i:
 *   S(t) = c0 + c1 dx + c2 dx^2 + c3 dx^3, dx = t - t_i,
 *   c0 = y_i, c1 = s_i, c2 = (3 delta_i - 2 s_i - s_{i+1})/h_i, c3 = (s_i + s_{i+1} - 2 delta_i)/h_i^2.
 *
 * Layout: y[n_t][n_sys] (systems fastest), coef[n_t-1][4][n_sys].  Returns 0, or -1 if n_t < 4, or -2 if t is
 * not strictly increasing.
 * ------------------------------------------------------------------------------------------------ */
#define DEFINE_SPLINE_FIT(NAME, T)                                                                   \
    int NAME(const double *t, const double *y, int n_t, int n_sys, T *coef)                          \
    {                                                                                                \
        int n = n_t, i, q;                                                                           \
        if (n < 4) return -1;                                                                        \
        for (i = 0; i + 1 < n; ++i)                                                                  \
            if (!(t[i + 1] > t[i])) return -2;                                                       \
        T *h = malloc(sizeof(T) * n), *dl = malloc(sizeof(T) * n);                                   \
        T *lo = malloc(sizeof(T) * n), *di = malloc(sizeof(T) * n), *up = malloc(sizeof(T) * n);     \
        T *rh = malloc(sizeof(T) * n), *s = malloc(sizeof(T) * n);                                   \
        for (i = 0; i + 1 < n; ++i) h[i] = (T)t[i + 1] - (T)t[i];                                    \
        for (q = 0; q < n_sys; ++q) {                                                                \
            for (i = 0; i + 1 < n; ++i)                                                              \
                dl[i] = ((T)y[(size_t)(i + 1) * n_sys + q] - (T)y[(size_t)i * n_sys + q]) / h[i];    \
            /* first row */                                                                          \
            lo[0] = 0; di[0] = h[1]; up[0] = h[0] + h[1];                                            \
            rh[0] = ((3 * h[0] + 2 * h[1]) * h[1] * dl[0] + h[0] * h[0] * dl[1]) / (h[0] + h[1]);    \
            for (i = 1; i <= n - 2; ++i) {                                                           \
                lo[i] = h[i]; di[i] = 2 * (h[i - 1] + h[i]); up[i] = h[i - 1];                       \
                rh[i] = 3 * (h[i] * dl[i - 1] + h[i - 1] * dl[i]);                                   \
            }                                                                                        \
            lo[n - 1] = h[n - 2] + h[n - 3]; di[n - 1] = h[n - 3]; up[n - 1] = 0;                    \
            rh[n - 1] = (h[n - 2] * h[n - 2] * dl[n - 3] +                                           \
                         (2 * h[n - 3] + 3 * h[n - 2]) * h[n - 3] * dl[n - 2]) / (h[n - 3] + h[n - 2]); \
            /* Thomas: forward elimination, back substitution */                                     \
            for (i = 1; i < n; ++i) {                                                                \
                T w = lo[i] / di[i - 1];                                                             \
                di[i] = di[i] - w * up[i - 1];                                                       \
                rh[i] = rh[i] - w * rh[i - 1];                                                       \
            }                                                                                        \
            s[n - 1] = rh[n - 1] / di[n - 1];                                                        \
            for (i = n - 2; i >= 0; --i) s[i] = (rh[i] - up[i] * s[i + 1]) / di[i];                  \
            for (i = 0; i + 1 < n; ++i) {                                                            \
                T *c = coef + (size_t)i * 4 * n_sys + q;                                             \
                c[0] = (T)y[(size_t)i * n_sys + q];                                                  \
                c[(size_t)n_sys] = s[i];                                                             \
                c[(size_t)2 * n_sys] = (3 * dl[i] - 2 * s[i] - s[i + 1]) / h[i];                     \
                c[(size_t)3 * n_sys] = (s[i] + s[i + 1] - 2 * dl[i]) / (h[i] * h[i]);                \
            }                                                                                        \
        }                                                                                            \
        free(h); free(dl); free(lo); free(di); free(up); free(rh); free(s);                          \
        return 0;                                                                                    \
    }

DEFINE_SPLINE_FIT(oracle_spline_fit, double)   /* amplitude systems: FP64 */
DEFINE_SPLINE_FIT(oracle_spline_fit_ext, ext)  /* phase systems: extended precision, R13 */

/* ------------------------------------------------------------------------------------------------
 * O2 -- spin-weighted spherical harmonic  sY_lm(theta, phi), used with s = -2 (Eq. (10):
 * "the regular -2 spin-weighted spherical harmonics").  The paper prints no formula; this is Goldberg et al.
 * (1967) Eq. (3.1) written with sin/cos half-angle powers so the poles are finite (R11):
 *   sY_lm = (-1)^m sqrt[ (l+m)!(l-m)!(2l+1) / (4 pi (l+s)!(l-s)!) ] e^{i m phi}
 *           * sum_r C(l-s, r) C(l+s, r+s-m) (-1)^{l-r-s} sin(th/2)^{2l-2r-s+m} cos(th/2)^{2r+s-m}
 * over r with 0 <= r <= l-s and 0 <= r+s-m <= l+s.  Returns 0, or -1 if l < |s| or |m| > l.
 * ------------------------------------------------------------------------------------------------ */
static ext factl(int k) { ext f = 1; for (int i = 2; i <= k; ++i) f *= i; return f; }
static ext binoml(int a, int b) { return (b < 0 || b > a) ? 0 : factl(a) / (factl(b) * factl(a - b)); }

int oracle_swsh(int s, int l, int m, double theta, double phi, double out[2])
{
    int as = s < 0 ? -s : s, am = m < 0 ? -m : m;
    if (l < as || am > l) return -1;
    ext pi = acosl(-1.0L);
    ext pref = sqrtl(factl(l + m) * factl(l - m) * (2 * l + 1) / (4 * pi * factl(l + s) * factl(l - s)));
    if (am % 2) pref = -pref;
    ext sh = sinl((ext)theta / 2), ch = cosl((ext)theta / 2), tot = 0;
    for (int r = 0; r <= l - s; ++r) {
        int k = r + s - m;
        if (k < 0 || k > l + s) continue;
        int ps = 2 * l - 2 * r - s + m, pc = 2 * r + s - m;
        ext term = binoml(l - s, r) * binoml(l + s, k);
        for (int i = 0; i < ps; ++i) term *= sh;
        for (int i = 0; i < pc; ++i) term *= ch;
        int e = l - r - s; if (e < 0) e = -e;
        tot += (e % 2) ? -term : term;
    }
    ext v = pref * tot;
    out[0] = (double)(v * cosl((ext)m * phi));
    out[1] = (double)(v * sinl((ext)m * phi));
    return 0;
}

int oracle_ylm(int l, int m, double theta, double phi, double out[2]) { return oracle_swsh(-2, l, m, theta, phi, out); }

/* ------------------------------------------------------------------------------------------------
 * O3 -- Mode Selector (sec. III D), sentence by sentence:
 *  "taking arrays of the power within each mode at each sparse time step determined from the complex
 *   amplitudes"            -> entries e with power P_e(k).  With harmonics ("combined with the
 *                             spin-weighted spherical harmonics and then put through mode selection") every
 *                             physical mode is its own entry: primary e = j, P = |A_j|^2 |Y+_j|^2, and for
 *                             m_j > 0 a mirror e = n_modes + rank(j), P = |A_j|^2 |Y-_j|^2, owned by j
 *                             (R4).  ylm_plus == NULL: primaries only, P = |A_j|^2.
 *  "operates entirely within each time step. It sorts the individual modes in descending order and computes
 *   a cumulative summation"-> per step: sort by P descending, equal P -> lower entry index first (R7);
 *                             inclusive cumulative sum C_r in extended precision.
 *  "where the additional power contributed by an individual mode falls below a user provided threshold
 *   related to the total power emitted (eps) at that time step (the final entry in the cumulative sum)"
 *                          -> total = C_last; rank 0 kept; rank r >= 1 kept iff C_{r-1} < (1-eps) total (R5).
 *  "the union of all contributing modes across all time steps" -> union over k of the owners; ascending j.
 *  eps <= 0 -> every mode kept, nothing sorted (R6).
 *
 * amp[n_t][n_modes][2]; ylm_*[n_modes][2]; keep_idx[n_modes] (padded with -1); margin[n_modes] (may be NULL):
 * min over steps and over the mode's entries of |C_{r-1} - (1-eps) total| / total, i.e. how close the mode ever
 * came to the threshold (INFINITY for rank-0-only / eps<=0) -- the parity test uses it for the north_star's
 * "within 1e-12 relative of the threshold" exception.
 * ------------------------------------------------------------------------------------------------ */
typedef struct { double p; int e; } sel_entry;

static int sel_cmp(const void *a, const void *b)
{
    const sel_entry *x = a, *y = b;
    if (x->p > y->p) return -1;
    if (x->p < y->p) return 1;
    return (x->e > y->e) - (x->e < y->e);
}

int oracle_select_modes(const double *amp, const int *m, const double *ylm_plus, const double *ylm_minus,
                        double eps, int n_t, int n_modes, int *keep_idx, int *n_keep, double *margin)
{
    int j, k, r, n_ent = n_modes;
    int *owner = malloc(sizeof(int) * 2 * (size_t)n_modes);
    char *keep = calloc((size_t)n_modes, 1);
    for (j = 0; j < n_modes; ++j) { owner[j] = j; if (margin) margin[j] = INFINITY; }
    if (ylm_plus)
        for (j = 0; j < n_modes; ++j)
            if (m[j] > 0) owner[n_ent++] = j;
    if (eps <= 0) {
        for (j = 0; j < n_modes; ++j) keep[j] = 1;
    } else {
        sel_entry *ent = malloc(sizeof(sel_entry) * (size_t)n_ent);
        for (k = 0; k < n_t; ++k) {
            const double *a = amp + (size_t)k * n_modes * 2;
            for (int e = 0; e < n_ent; ++e) {
                j = owner[e];
                double a2 = a[2 * j] * a[2 * j] + a[2 * j + 1] * a[2 * j + 1];
                double y2 = 1.0;
                if (ylm_plus) {
                    const double *y = (e < n_modes ? ylm_plus : ylm_minus) + 2 * (size_t)j;
                    y2 = y[0] * y[0] + y[1] * y[1];
                }
                ent[e].p = ylm_plus ? a2 * y2 : a2;
                ent[e].e = e;
            }
            qsort(ent, (size_t)n_ent, sizeof(sel_entry), sel_cmp); /* total order => stable by construction */
            ext total = 0;
            for (r = 0; r < n_ent; ++r) total += ent[r].p;          /* C_last */
            ext thr = (1.0L - (ext)eps) * total, c = 0;
            for (r = 0; r < n_ent; ++r) {                           /* c == C_{r-1} on entry */
                j = owner[ent[r].e];
                if (r == 0 || c < thr) keep[j] = 1;
                if (r >= 1 && margin && total > 0) {
                    double d = (double)(fabsl(c - thr) / total);
                    if (d < margin[j]) margin[j] = d;
                }
                c += ent[r].p;
            }
        }
        free(ent);
    }
    int cnt = 0;
    for (j = 0; j < n_modes; ++j) if (keep[j]) keep_idx[cnt++] = j;
    *n_keep = cnt;
    for (j = cnt; j < n_modes; ++j) keep_idx[j] = -1;
    free(owner); free(keep);
    return 0;
}

/* ------------------------------------------------------------------------------------------------
 * O4 -- interpolated summation (sec. III C; Eq. (9); Eq. (10)):
 *  "evaluates the spline at the sampling rate of the output data stream. Then, the output phase and amplitude
 *   values are combined within each mode according to Eq. (1) ... A_{l,-m,-k,-n} = (-1)^{l+k} A*_{lmkn} ...
 *   only compute modes for m >= 0; modes with m < 0 can be inferred ... the modes in a single time step are
 *   combined."
 *  h(t_i) = scale * sum_{j kept} [ Y+_j W_j + (m_j > 0) (-1)^{l_j} Y-_j conj(W_j) ],
 *  W_j = A_j(t_i) exp(-i (m_j Phi_phi(t_i) + n_j Phi_r(t_i))),  Y+ = -2Y_{l,m}, Y- = -2Y_{l,-m}   (k = 0, R9).
 *
 *  t_i = t0 + (i0+i)*dt, product and sum rounded separately (R14).  Outside [t_0, t_last] -> 0 (R12).
 *  Segment k = max{k : t_k <= t_i}, clamped to n_t-2; dx = t_i - t_k (one IEEE subtraction).
 *  Phases: extended-precision Horner with the extended coefficients of oracle_spline_fit_ext; theta_j in
 *  extended precision; cosl/sinl (glibc reduces the argument exactly) (R13, R15).
 *  Amplitudes: FP64 Horner of the FP64 coefficients.  Accumulation over j ascending in extended precision.
 *
 *  coef_amp[n_t-1][4][2*n_modes] (re, im interleaved per mode); coef_phase[n_t-1][4][2] (Phi_phi, Phi_r);
 *  keep_idx == NULL -> all n_modes modes; fold == 0 -> no mirror term (the list may then hold m < 0 entries, used
 *  by pin P5); h[n_samples][2] = (Re, Im) = (h_+, -h_x).
 * ------------------------------------------------------------------------------------------------ */
int oracle_sum_waveform(const double *t, const double *coef_amp, const ext *coef_phase,
                        const int *l, const int *m, const int *n, const int *keep_idx, int n_keep,
                        const double *ylm_plus, const double *ylm_minus, double scale, int fold,
                        double t0, double dt, long long i0, long long n_samples,
                        int n_t, int n_modes, double *h)
{
    if (n_t < 4) return -1;
    const int n_sys = 2 * n_modes;
    const int K = keep_idx ? n_keep : n_modes;
    long long i;
#pragma omp parallel for schedule(static)
    for (i = 0; i < n_samples; ++i) {
        double prod = (double)(i0 + i) * dt;
        double ti = t0 + prod;
        ext hr = 0, hi = 0;
        if (ti >= t[0] && ti <= t[n_t - 1]) {
            int lo = 0, hi_k = n_t - 1;          /* invariant: t[lo] <= ti, (hi_k == n_t-1 or t[hi_k] > ti) */
            while (hi_k - lo > 1) {
                int mid = (lo + hi_k) / 2;
                if (t[mid] <= ti) lo = mid; else hi_k = mid;
            }
            int k = lo > n_t - 2 ? n_t - 2 : lo;
            double dx = ti - t[k];
            const ext *cp = coef_phase + (size_t)k * 8;
            ext x = dx;
            ext Pphi = ((cp[6] * x + cp[4]) * x + cp[2]) * x + cp[0];
            ext Pr = ((cp[7] * x + cp[5]) * x + cp[3]) * x + cp[1];
            const double *ca = coef_amp + (size_t)k * 4 * n_sys;
            for (int q = 0; q < K; ++q) {
                int j = keep_idx ? keep_idx[q] : q;
                const double *c0 = ca + 2 * (size_t)j, *c1 = c0 + n_sys, *c2 = c1 + n_sys, *c3 = c2 + n_sys;
                double Ar = ((c3[0] * dx + c2[0]) * dx + c1[0]) * dx + c0[0];
                double Ai = ((c3[1] * dx + c2[1]) * dx + c1[1]) * dx + c0[1];
                ext th = (ext)m[j] * Pphi + (ext)n[j] * Pr;
                ext Er = cosl(th), Ei = -sinl(th);                       /* exp(-i theta) */
                ext Wr = (ext)Ar * Er - (ext)Ai * Ei, Wi = (ext)Ar * Ei + (ext)Ai * Er;
                ext yr = ylm_plus[2 * j], yi = ylm_plus[2 * j + 1];
                hr += yr * Wr - yi * Wi;
                hi += yr * Wi + yi * Wr;
                if (fold && m[j] > 0) {                                  /* Eq. (9), k = 0 */
                    ext sg = (l[j] % 2) ? -1.0L : 1.0L;
                    ext zr = sg * ylm_minus[2 * j], zi = sg * ylm_minus[2 * j + 1];
                    hr += zr * Wr + zi * Wi;                             /* Y- conj(W) */
                    hi += -zr * Wi + zi * Wr;
                }
            }
        }
        h[2 * i] = (double)(hr * scale);
        h[2 * i + 1] = (double)(hi * scale);
    }
    return 0;
}

/* ------------------------------------------------------------------------------------------------
 * O5 -- detector (solar-system-barycentre) frame, sec. II A, Eq. (4)-(8), and the mu/d_L
 * prefactor of Eq. (10).  NEXT-1 of SURVEY.md section 8(f).
 *  Eq. (4)  R = (sin qS cos phiS, sin qS sin phiS, cos qS)           line of sight to the source
 *  Eq. (5)  S = (sin qK cos phiK, sin qK sin phiK, cos qK)           MBH spin direction
 *  PAPER.md:96  "This convention leads to phi_src = -pi/2 always ... cos theta_src = -R.S"
 *  PAPER.md:98  "a rotation angle of pi/2 is applied. This rotation is equivalent to a phase shift of pi"
 *               -> factor e^{i pi} = -1
 *  PAPER.md:100 "The rotation to the solar system baricenter frame is twice the polarization angle, psi"
 *  Eq. (8)  prints psi = N/D with N = cos qS sin qK cos(phiS-phiK) - sin qS cos qK, D = sin qK sin(phiS-phiK):
 *           an angle equated to a ratio; the kludge construction the paper follows defines psi through its
 *           tangent, tan psi = N/D (R22).  psi = atan2(N, D); only 2 psi mod 2 pi enters, so the
 *           branch of the arctangent is immaterial.  N = D = 0 (S parallel to R, wave frame undefined): psi = 0.
 *  h_+^SSB - i h_x^SSB = e^{+2 i psi} (h_+ - i h_x): what the spin-2 combination h_+ - i h_x does when the polarisation
 *  basis is rotated by psi about the propagation direction z_w = -R, from the wave frame (x_w, y_w) of Eq. (6) to the
 *  right-handed pair (e_theta, -e_phi) at the sky position; Eq. (8)'s psi is exactly that angle (x_w = cos psi e_theta +
 *  sin psi e_phi), pinned geometrically in P12 (R22).
 * out[0] = theta_src, out[1] = phi_src, (out[2], out[3]) = factor = -(mu/d_L) e^{+2 i psi}.
 * All in extended precision, rounded once.
 * ------------------------------------------------------------------------------------------------ */
int oracle_frame(double qS, double phiS, double qK, double phiK, double mu_over_dl, double out[4])
{
    ext R[3] = { sinl((ext)qS) * cosl((ext)phiS), sinl((ext)qS) * sinl((ext)phiS), cosl((ext)qS) };
    ext S[3] = { sinl((ext)qK) * cosl((ext)phiK), sinl((ext)qK) * sinl((ext)phiK), cosl((ext)qK) };
    ext c = -(R[0] * S[0] + R[1] * S[1] + R[2] * S[2]);
    if (c > 1) c = 1;
    if (c < -1) c = -1;
    ext N = cosl((ext)qS) * sinl((ext)qK) * cosl((ext)phiS - (ext)phiK) - sinl((ext)qS) * cosl((ext)qK);
    ext D = sinl((ext)qK) * sinl((ext)phiS - (ext)phiK);
    ext psi = (N == 0 && D == 0) ? 0 : atan2l(N, D);
    out[0] = (double)acosl(c);
    out[1] = (double)(-acosl(-1.0L) / 2);
    out[2] = (double)(-(ext)mu_over_dl * cosl(2 * psi));
    out[3] = (double)(-(ext)mu_over_dl * sinl(2 * psi));
    return 0;
}

/* h_out = factor * h_in (complex), extended-precision products, rounded once. */
int oracle_frame_apply(const double *h_in, long long n, const double factor[2], double *h_out)
{
    for (long long i = 0; i < n; ++i) {
        ext a = h_in[2 * i], b = h_in[2 * i + 1], fr = factor[0], fi = factor[1];
        h_out[2 * i] = (double)(fr * a - fi * b);
        h_out[2 * i + 1] = (double)(fr * b + fi * a);
    }
    return 0;
}

/* ------------------------------------------------------------------------------------------------
 * O6 -- inner products with the PSD set to 1 (Eq. (15)-(17); "setting the PSD to 1 for all
 * frequencies to avoid noise-weighting").  NEXT-2 of SURVEY.md section 8(f).
 * Eq. (16) <a|b> = 4 Re int_0^inf conj(a~) b~ / S_n df.  With S_n = 1 and real a(t), b(t) sampled at dt, Parseval
 * gives <a|b> = 2 dt sum_i a_i b_i; the two polarisations of h = h_+ - i h_x are summed (R23), so for complex
 * series  <a|b> = 2 dt Re sum_i conj(a_i) b_i.  The imaginary part of the same sum is returned too (it is what a
 * phase-maximised overlap needs and costs nothing).
 * out[0] = <d|h>, out[1] = 2 dt Im sum conj(d_i) h_i, out[2] = <h|h>.  Sums in extended precision, index order.
 * ------------------------------------------------------------------------------------------------ */
int oracle_inner(const double *d, const double *h, long long n, double dt, double out[3])
{
    ext re = 0, im = 0, hh = 0;
    for (long long i = 0; i < n; ++i) {
        ext dr = d[2 * i], di = d[2 * i + 1], hr = h[2 * i], hi = h[2 * i + 1];
        re += dr * hr + di * hi;
        im += dr * hi - di * hr;
        hh += hr * hr + hi * hi;
    }
    out[0] = (double)(2 * (ext)dt * re);
    out[1] = (double)(2 * (ext)dt * im);
    out[2] = (double)(2 * (ext)dt * hh);
    return 0;
}

/* ------------------------------------------------------------------------------------------------
 * O7 -- direct summation (sec. III C: "performs a direct summation with amplitude and trajectory
 * information at the array density provided"; "combining the phase and amplitude information at
 * each time point in the data stream without interpolating any of these quantities").  NEXT-3 of SURVEY.md 8(f).
 *  h_i = scale * sum_j [ Y+_j W_ij + (m_j > 0) (-1)^{l_j} Y-_j conj(W_ij) ],
 *  W_ij = A_ij exp(-i (m_j Phi_phi,i + n_j Phi_r,i))      (Eq. (10) with the Eq. (9) fold)
 * amp[N][K][2] (modes fastest: the amplitude module's [n_t, n_modes] layout, at dense n_t = N);
 * phase[N][2] = (Phi_phi, Phi_r) in FP64 as given; the angle m Phi_phi + n Phi_r is formed and reduced in
 * extended precision (exact for the FP64 inputs to 2^-64 relative); accumulation over j in extended precision.
 * ------------------------------------------------------------------------------------------------ */
int oracle_sum_direct(const double *amp, const double *phase, const int *l, const int *m, const int *n,
                      const double *ylm_plus, const double *ylm_minus, double scale, int fold,
                      long long N, int K, double *h)
{
    long long i;
#pragma omp parallel for schedule(static)
    for (i = 0; i < N; ++i) {
        ext hr = 0, hi = 0;
        ext Pphi = phase[2 * i], Pr = phase[2 * i + 1];
        const double *a = amp + (size_t)i * K * 2;
        for (int j = 0; j < K; ++j) {
            ext th = (ext)m[j] * Pphi + (ext)n[j] * Pr;
            ext Er = cosl(th), Ei = -sinl(th);
            ext Wr = (ext)a[2 * j] * Er - (ext)a[2 * j + 1] * Ei, Wi = (ext)a[2 * j] * Ei + (ext)a[2 * j + 1] * Er;
            ext yr = ylm_plus[2 * j], yi = ylm_plus[2 * j + 1];
            hr += yr * Wr - yi * Wi;
            hi += yr * Wi + yi * Wr;
            if (fold && m[j] > 0) {
                ext sg = (l[j] % 2) ? -1.0L : 1.0L;
                ext zr = sg * ylm_minus[2 * j], zi = sg * ylm_minus[2 * j + 1];
                hr += zr * Wr + zi * Wi;
                hi += -zr * Wi + zi * Wr;
            }
        }
        h[2 * i] = (double)(hr * scale);
        h[2 * i + 1] = (double)(hi * scale);
    }
    return 0;
}

/* ------------------------------------------------------------------------------------------------
 * O8 -- interpolated summation with the polar index k and the third phase (generic Kerr shape), Eq. (1):
 * "Phi_mkn = m Phi_phi + k Phi_theta + n Phi_r", Eq. (19): with the spheroidal harmonics projected on
 * spherical ones "h = mu/d_L sum_lmkn A_lmkn(t) -2Y_lm(theta, phi) exp(-i Phi_mkn(t))", and Eq. (9) in full:
 * "A_{l,-m,-k,-n} = (-1)^{(l+k)} A*_lmkn".  NEXT-4 of SURVEY.md section 8(f).
 *  h(t_i) = scale * sum_{j kept} [ Y+_j W_j + (m_j > 0) (-1)^{l_j + k_j} Y-_j conj(W_j) ],
 *  W_j = A_j(t_i) exp(-i (m_j Phi_phi + k_j Phi_theta + n_j Phi_r)).
 * Everything else exactly as O4 (sample times, segment lookup, extended-precision phases, FP64 amplitudes, accumulation
 * order).  coef_phase[n_t-1][4][n_ph] with n_ph = 3: (Phi_phi, Phi_theta, Phi_r); n_ph = 2: (Phi_phi, Phi_r), k ignored
 * in the angle -- then the function is O4 apart from the fold sign, which is pinned against O4 with k = 0.
 * ------------------------------------------------------------------------------------------------ */
int oracle_sum_waveform_kerr(const double *t, const double *coef_amp, const ext *coef_phase, int n_ph,
                             const int *l, const int *m, const int *k, const int *n, const int *keep_idx, int n_keep,
                             const double *ylm_plus, const double *ylm_minus, double scale, int fold,
                             double t0, double dt, long long i0, long long n_samples,
                             int n_t, int n_modes, double *h)
{
    if (n_t < 4) return -1;
    if (n_ph != 2 && n_ph != 3) return -3;
    const int n_sys = 2 * n_modes;
    const int K = keep_idx ? n_keep : n_modes;
    long long i;
#pragma omp parallel for schedule(static)
    for (i = 0; i < n_samples; ++i) {
        double prod = (double)(i0 + i) * dt;
        double ti = t0 + prod;
        ext hr = 0, hi = 0;
        if (ti >= t[0] && ti <= t[n_t - 1]) {
            int lo = 0, hi_k = n_t - 1;
            while (hi_k - lo > 1) {
                int mid = (lo + hi_k) / 2;
                if (t[mid] <= ti) lo = mid; else hi_k = mid;
            }
            int seg = lo > n_t - 2 ? n_t - 2 : lo;
            double dx = ti - t[seg];
            const ext *cp = coef_phase + (size_t)seg * 4 * n_ph;
            ext x = dx, P[3] = {0, 0, 0};
            for (int q = 0; q < n_ph; ++q)
                P[q] = ((cp[3 * n_ph + q] * x + cp[2 * n_ph + q]) * x + cp[n_ph + q]) * x + cp[q];
            ext Pphi = P[0], Pth = n_ph == 3 ? P[1] : 0, Pr = n_ph == 3 ? P[2] : P[1];
            const double *ca = coef_amp + (size_t)seg * 4 * n_sys;
            for (int q = 0; q < K; ++q) {
                int j = keep_idx ? keep_idx[q] : q;
                const double *c0 = ca + 2 * (size_t)j, *c1 = c0 + n_sys, *c2 = c1 + n_sys, *c3 = c2 + n_sys;
                double Ar = ((c3[0] * dx + c2[0]) * dx + c1[0]) * dx + c0[0];
                double Ai = ((c3[1] * dx + c2[1]) * dx + c1[1]) * dx + c0[1];
                int kj = (n_ph == 3 && k) ? k[j] : 0;
                ext th = (ext)m[j] * Pphi + (ext)kj * Pth + (ext)n[j] * Pr;
                ext Er = cosl(th), Ei = -sinl(th);
                ext Wr = (ext)Ar * Er - (ext)Ai * Ei, Wi = (ext)Ar * Ei + (ext)Ai * Er;
                ext yr = ylm_plus[2 * j], yi = ylm_plus[2 * j + 1];
                hr += yr * Wr - yi * Wi;
                hi += yr * Wi + yi * Wr;
                if (fold && m[j] > 0) {                                  /* Eq. (9): (-1)^(l+k) */
                    int par = l[j] + (k ? k[j] : 0);
                    ext sg = (par % 2) ? -1.0L : 1.0L;
                    ext zr = sg * ylm_minus[2 * j], zi = sg * ylm_minus[2 * j + 1];
                    hr += zr * Wr + zi * Wi;
                    hi += -zr * Wi + zi * Wr;
                }
            }
        }
        h[2 * i] = (double)(hr * scale);
        h[2 * i + 1] = (double)(hi * scale);
    }
    return 0;
}
