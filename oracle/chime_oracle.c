/*
 * chime_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, double-precision CPU statement of what the CHIME/FRB hybrid
 * beamformer hot path computes (arXiv:1702.04728, PAPER.md).  Every transform is a
 * direct O(N^2) phase sum ("the interferometric phasing ... resembles
 * the functional form of a Fourier Transform"); there is no FFT, no blocking and no
 * reordering beyond the order the paper lists the steps in.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs may load this file.  It shares no code, table or constant with the CUDA path
 * under paper_1702_04728_b200/csrc/.
 *
 * Steps (notation of DESIGN.md section "The path"):
 *   1. unpack     x = (b>>4)-8 + i((b&15)-8)                 PAPER.md:40-41,47; reading A1
 *   2. gains      v = g * x                                  BASELINE.json (not in paper); A16
 *   3. N-S        Y[m] = sum_n v[n] exp(-2 pi i J[m] n / NP) PAPER.md:59-61 (zero-padded DFT,
 *                                                            nearest-bin selection)
 *   4. E-W        Z[e] = sum_cyl exp(-2 pi i f x_cyl sin(phi_e)/c0) Y[cyl]
 *   5. upchan     S[q] = sum_u Z[U r + u] exp(-2 pi i q u / U)
 *   6. detect     I[g] = norm * sum_{r<n_int} sum_pol sum_{q in group g} |S|^2
 *                                                            PAPER.md:37-39,42,53; A9-A12
 *   7. quantise   q = clamp(rne(I*scale + offset), 0, 255)   PAPER.md:40,53; A11
 *   index table   J[m] = rhu(P (m - N/2) f / f_ref) mod NP   PAPER.md:61,67,75-78 eq.(1),(2); A2-A4
 *
 * Pins (tests/test_oracle_pins.py): brute force with literal cexp on tiny arrays, numpy.fft
 * special cases, the closed-form Dirichlet response to a tone, Parseval, linearity,
 * zero-in/zero-out, single-input impulse, Table 1 arithmetic, the alias geometry the paper
 * prints in section 3.3, index-table invariants.
 * PARITY UNPINNED (conventions the paper does not fix):
 *   A1 nibble order/offset encoding, A9 order of the 16 fine channels, A11 the intensity
 *   normalisation 1/(N N_c U) and the u8 scale/offset, A2 the default f_ref = 600 MHz.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_C0 299792458.0 /* speed of light, m/s (eq. (1),(2): "c") */
static const double ORACLE_PI = 3.14159265358979323846264338327950288;

typedef struct { double re, im; } cplx;

static inline cplx cmul(cplx a, cplx b) {
    cplx r = { a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re };
    return r;
}

int oracle_max_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* round-half-up: floor(x) + [frac >= 0.5]  (eq. (1): "+ 0.5" then integer part; reading A3) */
static long rhu(double x) {
    double fl = floor(x);
    return (long)fl + ((x - fl) >= 0.5 ? 1 : 0);
}

static int32_t mod_np(long j, int np) {
    long r = j % np;
    if (r < 0) r += np;
    return (int32_t)r;
}

/*
 * Index table of the clamped N-S beams, eq. (1)+(2) with the desired pointings on the
 * native n_feed-point grid at f_ref (reading A2):  sin(theta_m) = (m - N/2) c / (N d f_ref).
 * Substituted in eq. (1)+(2):  t_m + dt_m = P (m - N/2) f / f_ref + 0.5; d and c cancel.
 * Evaluation order pinned (A3): one multiply of an exact integer by f, one division.
 */
void oracle_ns_index(int n_feed, int np, double f_mhz, double fref_mhz, int32_t *J) {
    int P = np / n_feed;
    for (int m = 0; m < n_feed; ++m) {
        double k = (double)(P * (m - n_feed / 2));
        double x = (k * f_mhz) / fref_mhz;
        J[m] = mod_np(rhu(x), np);
    }
}

/* Same table for an explicit list of desired pointings sin(theta_m): eq. (1)+(2) as printed,
 * t = N P f (d/c) sin(theta) + 0.5, integer part, mod NP. */
void oracle_ns_index_sintheta(int n_feed, int np, double f_mhz, double feed_spacing_m,
                              const double *sin_theta, int n_beam, int32_t *J) {
    for (int m = 0; m < n_beam; ++m) {
        double x = (double)np * (f_mhz * 1e6) * (feed_spacing_m / ORACLE_C0) * sin_theta[m];
        J[m] = mod_np(rhu(x), np);
    }
    (void)n_feed;
}

/* Step 1. out[2i] = real, out[2i+1] = imag. */
void oracle_unpack(const uint8_t *b, size_t n, int8_t *out) {
    for (size_t i = 0; i < n; ++i) {
        out[2 * i] = (int8_t)((int)(b[i] >> 4) - 8);
        out[2 * i + 1] = (int8_t)((int)(b[i] & 15) - 8);
    }
}

/* E-W weights, step 4: w[e][cyl] = exp(-2 pi i f (cyl * spacing) sin(phi_e) / c0). */
void oracle_ew_weights(int n_cyl, int n_ew, double f_mhz, double cyl_spacing_m,
                       const double *ew_deg, double *w /* [n_ew][n_cyl][2] */) {
    for (int e = 0; e < n_ew; ++e)
        for (int c = 0; c < n_cyl; ++c) {
            double s = sin(ew_deg[e] * ORACLE_PI / 180.0);
            double ph = -2.0 * ORACLE_PI * (f_mhz * 1e6) * ((double)c * cyl_spacing_m) * s / ORACLE_C0;
            w[2 * (e * n_cyl + c)] = cos(ph);
            w[2 * (e * n_cyl + c) + 1] = sin(ph);
        }
}

/*
 * Steps 2-4 for a block of time samples: voltages in, beamformed voltages out.
 *   x  [n_t][n_pol][n_cyl][n_feed] complex (re,im interleaved doubles)
 *   g  [n_pol][n_cyl][n_feed]      complex
 *   J  [n_beam]                    selected bin per N-S beam
 *   Z  [n_t][n_pol][n_ew][n_beam]  complex out   (the paper's kernel-1 output order)
 */
void oracle_beamform(const double *x, const double *g, int n_t, int n_pol, int n_cyl, int n_feed,
                     int np, const int32_t *J, int n_beam, int n_ew, const double *w_ew, double *Z) {
    cplx *tw = (cplx *)malloc(sizeof(cplx) * (size_t)np);
    for (int k = 0; k < np; ++k) {
        double ph = -2.0 * ORACLE_PI * (double)k / (double)np;
        tw[k].re = cos(ph);
        tw[k].im = sin(ph);
    }
    const cplx *X = (const cplx *)x;
    const cplx *G = (const cplx *)g;
    const cplx *W = (const cplx *)w_ew;
    cplx *Zc = (cplx *)Z;
#pragma omp parallel
    {
        cplx *v = (cplx *)malloc(sizeof(cplx) * (size_t)n_cyl * n_feed);
        cplx *Y = (cplx *)malloc(sizeof(cplx) * (size_t)n_cyl * n_beam);
#pragma omp for collapse(2) schedule(static)
        for (int t = 0; t < n_t; ++t)
            for (int p = 0; p < n_pol; ++p) {
                const cplx *xr = X + ((size_t)t * n_pol + p) * n_cyl * n_feed;
                const cplx *gr = G + (size_t)p * n_cyl * n_feed;
                /* step 2 */
                for (int i = 0; i < n_cyl * n_feed; ++i) v[i] = cmul(gr[i], xr[i]);
                /* step 3: direct sum over feeds for every selected bin */
                for (int c = 0; c < n_cyl; ++c)
                    for (int m = 0; m < n_beam; ++m) {
                        cplx acc = { 0.0, 0.0 };
                        long j = J[m];
                        for (int n = 0; n < n_feed; ++n) {
                            cplx pr = cmul(v[c * n_feed + n], tw[(j * n) % np]);
                            acc.re += pr.re;
                            acc.im += pr.im;
                        }
                        Y[c * n_beam + m] = acc;
                    }
                /* step 4 */
                for (int e = 0; e < n_ew; ++e)
                    for (int m = 0; m < n_beam; ++m) {
                        cplx acc = { 0.0, 0.0 };
                        for (int c = 0; c < n_cyl; ++c) {
                            cplx pr = cmul(W[e * n_cyl + c], Y[c * n_beam + m]);
                            acc.re += pr.re;
                            acc.im += pr.im;
                        }
                        Zc[(((size_t)t * n_pol + p) * n_ew + e) * n_beam + m] = acc;
                    }
            }
        free(v);
        free(Y);
    }
    free(tw);
}

/* Step 3 alone, every one of the NP bins (used by the Parseval pin). */
void oracle_ns_dft_allbins(const double *v, int n_feed, int np, double *Y /* [np] complex */) {
    const cplx *V = (const cplx *)v;
    cplx *Yc = (cplx *)Y;
    for (int j = 0; j < np; ++j) {
        cplx acc = { 0.0, 0.0 };
        for (int n = 0; n < n_feed; ++n) {
            double ph = -2.0 * ORACLE_PI * (double)(((long)j * n) % np) / (double)np;
            cplx t = { cos(ph), sin(ph) };
            cplx pr = cmul(V[n], t);
            acc.re += pr.re;
            acc.im += pr.im;
        }
        Yc[j] = acc;
    }
}

/*
 * Steps 5-6 for one output cell: Z [n_int*U][n_pol][n_beams] complex in,
 * I [n_beams][n_fine] out.  Rectangular window, non-overlapping blocks (A8);
 * group g = ((q + U/2) mod U) div D, D = U / n_fine (A9); norm multiplies the sum (A11).
 * If S_out != NULL it receives S [n_int][U][n_pol][n_beams] complex (for the Parseval pin).
 */
void oracle_upchan_detect(const double *Z, int n_int, int U, int n_pol, int n_beams, int n_fine,
                          double norm, double *I, double *S_out) {
    cplx *tw = (cplx *)malloc(sizeof(cplx) * (size_t)U);
    for (int k = 0; k < U; ++k) {
        double ph = -2.0 * ORACLE_PI * (double)k / (double)U;
        tw[k].re = cos(ph);
        tw[k].im = sin(ph);
    }
    const cplx *Zc = (const cplx *)Z;
    cplx *Sc = (cplx *)S_out;
    int D = U / n_fine;
#pragma omp parallel for schedule(static)
    for (int b = 0; b < n_beams; ++b) {
        for (int gq = 0; gq < n_fine; ++gq) I[(size_t)b * n_fine + gq] = 0.0;
        for (int r = 0; r < n_int; ++r)
            for (int p = 0; p < n_pol; ++p)
                for (int q = 0; q < U; ++q) {
                    cplx acc = { 0.0, 0.0 };
                    for (int u = 0; u < U; ++u) {
                        cplx z = Zc[(((size_t)(U * r + u)) * n_pol + p) * n_beams + b];
                        cplx pr = cmul(z, tw[((long)q * u) % U]);
                        acc.re += pr.re;
                        acc.im += pr.im;
                    }
                    if (Sc) Sc[(((size_t)r * U + q) * n_pol + p) * n_beams + b] = acc;
                    int gq = ((q + U / 2) % U) / D;
                    I[(size_t)b * n_fine + gq] += acc.re * acc.re + acc.im * acc.im;
                }
        for (int gq = 0; gq < n_fine; ++gq) I[(size_t)b * n_fine + gq] *= norm;
    }
    free(tw);
}

/* Step 7.  rint() under the default rounding mode is round-half-to-even. */
void oracle_quantize(const double *I, size_t n, double scale, double offset, uint8_t *out) {
    for (size_t i = 0; i < n; ++i) {
        double q = rint(I[i] * scale + offset);
        if (q < 0.0) q = 0.0;
        if (q > 255.0) q = 255.0;
        out[i] = (uint8_t)q;
    }
}

/*
 * One output cell from voltages (float hook used by the closed-form pins):
 * steps 2-6 in order.  I_out [n_ew][n_beam][n_fine]; norm = 1/(n_feed n_cyl U) (A11).
 */
void oracle_cell_from_voltage(const double *x, const double *g, int n_pol, int n_cyl, int n_feed,
                              int np, const int32_t *J, int n_beam, int n_ew, const double *w_ew,
                              int U, int n_int, int n_fine, double *I_out) {
    int n_t = n_int * U;
    size_t nz = (size_t)n_t * n_pol * n_ew * n_beam;
    double *Z = (double *)malloc(sizeof(double) * 2 * nz);
    oracle_beamform(x, g, n_t, n_pol, n_cyl, n_feed, np, J, n_beam, n_ew, w_ew, Z);
    double norm = 1.0 / ((double)n_feed * (double)n_cyl * (double)U);
    oracle_upchan_detect(Z, n_int, U, n_pol, n_ew * n_beam, n_fine, norm, I_out, NULL);
    free(Z);
}

/*
 * One output cell from packed baseband (steps 1-6):
 *   in_u8  [n_int*U][n_pol*n_cyl*n_feed] bytes, input index i = (pol*n_cyl + cyl)*n_feed + feed
 *   gains  [n_pol*n_cyl*n_feed][2] float32 (the values the plan is given), or NULL = unit
 */
void oracle_cell_from_u8(const uint8_t *in_u8, const float *gains, int n_pol, int n_cyl, int n_feed,
                         int np, const int32_t *J, int n_beam, int n_ew, const double *w_ew, int U,
                         int n_int, int n_fine, double *I_out) {
    int n_t = n_int * U;
    size_t n_in = (size_t)n_pol * n_cyl * n_feed;
    double *x = (double *)malloc(sizeof(double) * 2 * n_t * n_in);
    double *g = (double *)malloc(sizeof(double) * 2 * n_in);
    for (size_t i = 0; i < (size_t)n_t * n_in; ++i) {
        int8_t ri[2];
        oracle_unpack(in_u8 + i, 1, ri);
        x[2 * i] = (double)ri[0];
        x[2 * i + 1] = (double)ri[1];
    }
    for (size_t i = 0; i < n_in; ++i) {
        g[2 * i] = gains ? (double)gains[2 * i] : 1.0;
        g[2 * i + 1] = gains ? (double)gains[2 * i + 1] : 0.0;
    }
    oracle_cell_from_voltage(x, g, n_pol, n_cyl, n_feed, np, J, n_beam, n_ew, w_ew, U, n_int,
                             n_fine, I_out);
    free(x);
    free(g);
}

/*
 * Exact chromatic alignment (section 4: "beam interpolation, which would enable the
 * FFT-formed beams to be perfectly aligned across observing frequencies"; added after the steps
 * above, which it leaves untouched).  Step 3 with the nearest-bin phase J[m] n / NP replaced by
 * the phase of the desired pointing itself:
 *     Y[m] = sum_n v[n] exp(-2 pi i n turns[m]),   turns[m] = f d sin(theta_m) / c0
 * (cycles of phase per feed; for the native grid of reading A2, turns[m] = (m - N/2) f / (N f_ref)).
 * Everything else (steps 2, 4) as in oracle_beamform.  The argument n * turns is reduced to
 * [-1/2, 1/2) before cos/sin.
 */
void oracle_beamform_exact(const double *x, const double *g, int n_t, int n_pol, int n_cyl,
                           int n_feed, const double *turns, int n_beam, int n_ew,
                           const double *w_ew, double *Z) {
    cplx *tw = (cplx *)malloc(sizeof(cplx) * (size_t)n_beam * n_feed);
    for (int m = 0; m < n_beam; ++m)
        for (int n = 0; n < n_feed; ++n) {
            double ph = (double)n * turns[m];
            ph -= floor(ph + 0.5);
            tw[(size_t)m * n_feed + n].re = cos(-2.0 * ORACLE_PI * ph);
            tw[(size_t)m * n_feed + n].im = sin(-2.0 * ORACLE_PI * ph);
        }
    const cplx *X = (const cplx *)x;
    const cplx *G = (const cplx *)g;
    const cplx *W = (const cplx *)w_ew;
    cplx *Zc = (cplx *)Z;
#pragma omp parallel for collapse(2) schedule(static)
    for (int t = 0; t < n_t; ++t)
        for (int p = 0; p < n_pol; ++p) {
            const cplx *xr = X + ((size_t)t * n_pol + p) * n_cyl * n_feed;
            const cplx *gr = G + (size_t)p * n_cyl * n_feed;
            for (int e = 0; e < n_ew; ++e)
                for (int m = 0; m < n_beam; ++m) {
                    cplx z = { 0.0, 0.0 };
                    for (int c = 0; c < n_cyl; ++c) {
                        cplx y = { 0.0, 0.0 };
                        for (int n = 0; n < n_feed; ++n) {
                            cplx pr = cmul(cmul(gr[c * n_feed + n], xr[c * n_feed + n]),
                                           tw[(size_t)m * n_feed + n]);
                            y.re += pr.re;
                            y.im += pr.im;
                        }
                        cplx pr = cmul(W[e * n_cyl + c], y);
                        z.re += pr.re;
                        z.im += pr.im;
                    }
                    Zc[(((size_t)t * n_pol + p) * n_ew + e) * n_beam + m] = z;
                }
        }
    free(tw);
}

/* One output cell from packed baseband with exact pointing: steps 1, 2, 3 (exact), 4, 5, 6. */
void oracle_cell_from_u8_exact(const uint8_t *in_u8, const float *gains, int n_pol, int n_cyl,
                               int n_feed, const double *turns, int n_beam, int n_ew,
                               const double *w_ew, int U, int n_int, int n_fine, double *I_out) {
    int n_t = n_int * U;
    size_t n_in = (size_t)n_pol * n_cyl * n_feed;
    double *x = (double *)malloc(sizeof(double) * 2 * n_t * n_in);
    double *g = (double *)malloc(sizeof(double) * 2 * n_in);
    for (size_t i = 0; i < (size_t)n_t * n_in; ++i) {
        int8_t ri[2];
        oracle_unpack(in_u8 + i, 1, ri);
        x[2 * i] = (double)ri[0];
        x[2 * i + 1] = (double)ri[1];
    }
    for (size_t i = 0; i < n_in; ++i) {
        g[2 * i] = gains ? (double)gains[2 * i] : 1.0;
        g[2 * i + 1] = gains ? (double)gains[2 * i + 1] : 0.0;
    }
    size_t nz = (size_t)n_t * n_pol * n_ew * n_beam;
    double *Z = (double *)malloc(sizeof(double) * 2 * nz);
    oracle_beamform_exact(x, g, n_t, n_pol, n_cyl, n_feed, turns, n_beam, n_ew, w_ew, Z);
    double norm = 1.0 / ((double)n_feed * (double)n_cyl * (double)U);
    oracle_upchan_detect(Z, n_int, U, n_pol, n_ew * n_beam, n_fine, norm, I_out, NULL);
    free(Z);
    free(x);
    free(g);
}
