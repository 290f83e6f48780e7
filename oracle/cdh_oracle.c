/*
 * cdh_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, obviously-correct CPU oracle for the particle-pair distance histogram of
 * Reuter & Koefinger, "CADISHI" (arxiv 1808.01478).  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may call it.  It shares no code with the CUDA
 * library under paper_1808_01478_b200/csrc/ and includes none of its headers.
 *
 * What it computes is the paper's plain definition, written out as the double loop of
 *   Algorithm 1 (section 2.2): for i in species 1, for j in species 2:
 *       distance vector, minimum image (periodic only), r = sqrt(x^2+y^2+z^2),
 *       kappa = (int) n_bins * r / r_max, ++hist[kappa];
 *   the single-species variant starts the inner loop at j = i + 1;
 *   bins are half open, r_kappa <= r < r_kappa + dr (Eq. 4);
 *   minimum image dx' = dx - b nint(b^-1 dx) (Eq. 5), b diagonal for an
 *   orthorhombic box; for a triclinic box the Eq.-5 vector is additionally shifted
 *   to the neighbouring cells and the minimum taken ("three-fold loop over all neighbouring
 *   boxes");
 *   counts are integers, 64 bit in the result;
 *   histograms of all frames of a call are summed (Eq. 2, sum over k).
 *
 * The result is made bit-reproducible by pinning ONE IEEE-754 operation sequence (DESIGN.md
 * "Pinned sequence"): every operation below is individually rounded in T
 * (float for the fp32 oracle, double for the fp64 oracle); there is no FMA contraction (compile
 * with -ffp-contract=off -fno-fast-math), sqrt is correctly rounded, nint is rint() in the default
 * round-half-to-even mode (the paper's CPU code uses nearbyint()).
 *
 * Readings of the paper where it is silent (numbers as in SURVEY.md 8c):
 *   Q1 scale = (T)((double)n_bins / r_max) precomputed, bin = floor(r * scale);
 *   Q2 pairs with !(r < (T)r_max) are dropped in every box mode;
 *   Q3 a kept pair whose r*scale rounds up to n_bins goes to bin n_bins-1;
 *   Q4 floor => lower bin edge inclusive;  Q5 nint ties to even;
 *   Q6 API box rows are the box vectors, mathematical b has them as columns;
 *   Q7/Q8 triclinic: Eq. 5 first, then ALWAYS the minimum over the 27 shifts i*a+j*b+k*c,
 *         i,j,k in {-1,0,1};  Q10 unique unordered pairs, self excluded.
 *
 * Parity pins (tests/test_oracle_pins.py, -m "not gpu"): total counts N(N-1)/2 and N1*N2, the
 * hand-computed 4-particle examples in tests/golden/, 125-image brute force on tiny dyadic
 * periodic boxes, permutation / species-swap symmetry, numpy reduction in the non-periodic case,
 * ideal-gas shell counts, the > 2^32 single-bin case; for cdh_oracle_rdf (tests/test_oracle_rdf.py): the ideal gas
 * g = 1, a simple-cubic crystal's peaks and coordination numbers, the bin-centre shell identity, scaling laws.
 *
 * Threads: OpenMP over the outer particle loop with thread-private uint64 histograms summed at the
 * end (integer sums are order free).  This is for wall time only.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define CDHO_BOX_NONE 0
#define CDHO_BOX_ORTHO 1
#define CDHO_BOX_TRICLINIC 2

/* Double-precision derivation of b (columns = box vectors) and b^-1 = adj(b)/det(b) with the
 * fixed parenthesisation of DESIGN.md "Host-derived constants".  box9 rows are the box vectors. */
static void derive_b_and_inverse(const double *box9, double B[3][3], double Binv[3][3])
{
    for (int r = 0; r < 3; ++r)
        for (int c = 0; c < 3; ++c)
            B[r][c] = box9[c * 3 + r];
    const double det = B[0][0] * (B[1][1] * B[2][2] - B[1][2] * B[2][1])
                     - B[0][1] * (B[1][0] * B[2][2] - B[1][2] * B[2][0])
                     + B[0][2] * (B[1][0] * B[2][1] - B[1][1] * B[2][0]);
    /* Binv[r][c] = cofactor(c, r) / det, each 2x2 cofactor written (p*q - r*s). */
    Binv[0][0] =  (B[1][1] * B[2][2] - B[1][2] * B[2][1]) / det;
    Binv[0][1] = -(B[0][1] * B[2][2] - B[0][2] * B[2][1]) / det;
    Binv[0][2] =  (B[0][1] * B[1][2] - B[0][2] * B[1][1]) / det;
    Binv[1][0] = -(B[1][0] * B[2][2] - B[1][2] * B[2][0]) / det;
    Binv[1][1] =  (B[0][0] * B[2][2] - B[0][2] * B[2][0]) / det;
    Binv[1][2] = -(B[0][0] * B[1][2] - B[0][2] * B[1][0]) / det;
    Binv[2][0] =  (B[1][0] * B[2][1] - B[1][1] * B[2][0]) / det;
    Binv[2][1] = -(B[0][0] * B[2][1] - B[0][1] * B[2][0]) / det;
    Binv[2][2] =  (B[0][0] * B[1][1] - B[0][1] * B[1][0]) / det;
}

/* ------------------------------------------------------------------------------------------ */
/* The generic body is instantiated twice by textual inclusion of the macro below: T = float   */
/* and T = double.  SQRT / RINT / FLOOR are the matching libm routines.                        */
/* ------------------------------------------------------------------------------------------ */
#define CDHO_DEFINE(T, SUF, SQRT, RINT, FLOOR)                                                     \
                                                                                                   \
typedef struct {                                                                                   \
    int box_type;                                                                                  \
    T L[3], invL[3];            /* ORTHO */                                                        \
    T B[3][3], Binv[3][3];      /* TRICLINIC, columns of B = box vectors */                        \
    T S[27][3];                 /* TRICLINIC shift vectors */                                      \
} box_##SUF;                                                                                       \
                                                                                                   \
static void box_setup_##SUF(box_##SUF *bx, int box_type, const double *box9)                       \
{                                                                                                  \
    memset(bx, 0, sizeof *bx);                                                                     \
    bx->box_type = box_type;                                                                       \
    if (box_type == CDHO_BOX_ORTHO) {                                                              \
        for (int c = 0; c < 3; ++c) {                                                              \
            bx->L[c] = (T)box9[c * 3 + c];                                                         \
            bx->invL[c] = (T)(1.0 / box9[c * 3 + c]);                                              \
        }                                                                                          \
    } else if (box_type == CDHO_BOX_TRICLINIC) {                                                   \
        double B[3][3], Bi[3][3];                                                                  \
        derive_b_and_inverse(box9, B, Bi);                                                         \
        for (int r = 0; r < 3; ++r)                                                                \
            for (int c = 0; c < 3; ++c) {                                                          \
                bx->B[r][c] = (T)B[r][c];                                                          \
                bx->Binv[r][c] = (T)Bi[r][c];                                                      \
            }                                                                                      \
        int m = 0;                                                                                 \
        for (int i = -1; i <= 1; ++i)                                                              \
            for (int j = -1; j <= 1; ++j)                                                          \
                for (int k = -1; k <= 1; ++k, ++m)                                                 \
                    for (int r = 0; r < 3; ++r)                                                    \
                        bx->S[m][r] = ((T)i * bx->B[r][0] + (T)j * bx->B[r][1])                    \
                                      + (T)k * bx->B[r][2];                                        \
    }                                                                                              \
}                                                                                                  \
                                                                                                   \
/* Squared minimum-image distance of one pair, the pinned sequence. */                            \
static inline T pair_d2_##SUF(const box_##SUF *bx, T xi, T yi, T zi, T xj, T yj, T zj)             \
{                                                                                                  \
    T dx = xj - xi, dy = yj - yi, dz = zj - zi;                                                    \
    if (bx->box_type == CDHO_BOX_ORTHO) {                                                          \
        T t, n;                                                                                    \
        t = dx * bx->invL[0]; n = RINT(t); dx = dx - bx->L[0] * n;                                 \
        t = dy * bx->invL[1]; n = RINT(t); dy = dy - bx->L[1] * n;                                 \
        t = dz * bx->invL[2]; n = RINT(t); dz = dz - bx->L[2] * n;                                 \
    } else if (bx->box_type == CDHO_BOX_TRICLINIC) {                                               \
        T s[3], n[3], e[3];                                                                        \
        const T d[3] = {dx, dy, dz};                                                               \
        for (int k = 0; k < 3; ++k) {                                                              \
            s[k] = (bx->Binv[k][0] * dx + bx->Binv[k][1] * dy) + bx->Binv[k][2] * dz;              \
            n[k] = RINT(s[k]);                                                                     \
        }                                                                                          \
        for (int r = 0; r < 3; ++r) {                                                              \
            T sh = (bx->B[r][0] * n[0] + bx->B[r][1] * n[1]) + bx->B[r][2] * n[2];                 \
            e[r] = d[r] - sh;                                                                      \
        }                                                                                          \
        T best = (T)INFINITY;                                                                      \
        for (int m = 0; m < 27; ++m) {                                                             \
            T cx = e[0] + bx->S[m][0], cy = e[1] + bx->S[m][1], cz = e[2] + bx->S[m][2];           \
            T c2 = (cx * cx + cy * cy) + cz * cz;                                                  \
            if (c2 < best) best = c2;                                                              \
        }                                                                                          \
        return best;                                                                               \
    }                                                                                              \
    return (dx * dx + dy * dy) + dz * dz;                                                          \
}                                                                                                  \
                                                                                                   \
/* One species pair of one frame into hist (uint64[n_bins]).  xi/xj: AoS xyz of element type C    \
 * (the stored coordinate type), converted to T on load (float->double is exact). */              \
static void species_pair_##SUF(const box_##SUF *bx, const void *ci_, int ni, const void *cj_,      \
                               int nj, int same, int coords_f64, T rmax, T scale, int n_bins,      \
                               uint64_t *hist)                                                     \
{                                                                                                  \
    _Pragma("omp parallel")                                                                        \
    {                                                                                              \
        uint64_t *priv = (uint64_t *)calloc((size_t)n_bins, sizeof(uint64_t));                     \
        _Pragma("omp for schedule(dynamic, 16)")                                                   \
        for (int i = 0; i < ni; ++i) {                                                             \
            T xi, yi, zi;                                                                          \
            if (coords_f64) { const double *c = (const double *)ci_ + 3 * (size_t)i;               \
                              xi = (T)c[0]; yi = (T)c[1]; zi = (T)c[2]; }                          \
            else            { const float  *c = (const float  *)ci_ + 3 * (size_t)i;               \
                              xi = (T)c[0]; yi = (T)c[1]; zi = (T)c[2]; }                          \
            for (int j = same ? i + 1 : 0; j < nj; ++j) {                                          \
                T xj, yj, zj;                                                                      \
                if (coords_f64) { const double *c = (const double *)cj_ + 3 * (size_t)j;           \
                                  xj = (T)c[0]; yj = (T)c[1]; zj = (T)c[2]; }                      \
                else            { const float  *c = (const float  *)cj_ + 3 * (size_t)j;           \
                                  xj = (T)c[0]; yj = (T)c[1]; zj = (T)c[2]; }                      \
                const T d2 = pair_d2_##SUF(bx, xi, yi, zi, xj, yj, zj);                            \
                const T d = SQRT(d2);                                                              \
                if (!(d < rmax)) continue;          /* drops d >= r_max and NaN */                 \
                int64_t bin = (int64_t)FLOOR(d * scale);                                           \
                if (bin > n_bins - 1) bin = n_bins - 1;                                            \
                priv[bin] += 1;                                                                    \
            }                                                                                      \
        }                                                                                          \
        _Pragma("omp critical")                                                                    \
        for (int b = 0; b < n_bins; ++b) hist[b] += priv[b];                                       \
        free(priv);                                                                                \
    }                                                                                              \
}                                                                                                  \
                                                                                                   \
static int histograms_##SUF(const void *coords, int coords_f64, int n_frames,                      \
                            const int32_t *species_offsets, int n_species, int box_type,           \
                            const double *box, int n_boxes, double r_max, int n_bins,              \
                            uint64_t *out)                                                         \
{                                                                                                  \
    const size_t n_total = (size_t)species_offsets[n_species];                                     \
    const size_t esz = coords_f64 ? sizeof(double) : sizeof(float);                                \
    const T rmax_T = (T)r_max;                                                                     \
    const T scale_T = (T)((double)n_bins / r_max);                                                 \
    const int n_hist = n_species * (n_species + 1) / 2;                                            \
    memset(out, 0, (size_t)n_hist * (size_t)n_bins * sizeof(uint64_t));                           \
    for (int f = 0; f < n_frames; ++f) {                                                           \
        box_##SUF bx;                                                                              \
        box_setup_##SUF(&bx, box_type, box_type == CDHO_BOX_NONE ? NULL                            \
                                       : box + 9 * (size_t)(n_boxes == 1 ? 0 : f));                \
        const char *frame = (const char *)coords + (size_t)f * n_total * 3 * esz;                  \
        int h = 0;                                                                                 \
        for (int p = 0; p < n_species; ++p)                                                        \
            for (int q = p; q < n_species; ++q, ++h) {                                             \
                const int ni = species_offsets[p + 1] - species_offsets[p];                        \
                const int nj = species_offsets[q + 1] - species_offsets[q];                        \
                species_pair_##SUF(&bx, frame + (size_t)species_offsets[p] * 3 * esz, ni,          \
                                   frame + (size_t)species_offsets[q] * 3 * esz, nj, p == q,       \
                                   coords_f64, rmax_T, scale_T, n_bins,                            \
                                   out + (size_t)h * (size_t)n_bins);                              \
            }                                                                                      \
    }                                                                                              \
    return 0;                                                                                      \
}                                                                                                  \
                                                                                                   \
static double single_pair_d2_##SUF(const double *pi, const double *pj, int box_type,               \
                                   const double *box9)                                             \
{                                                                                                  \
    box_##SUF bx;                                                                                  \
    box_setup_##SUF(&bx, box_type, box9);                                                          \
    return (double)pair_d2_##SUF(&bx, (T)pi[0], (T)pi[1], (T)pi[2], (T)pj[0], (T)pj[1], (T)pj[2]); \
}

CDHO_DEFINE(float, f32, sqrtf, rintf, floorf)
CDHO_DEFINE(double, f64, sqrt, rint, floor)

/* ------------------------------- exported entry points ------------------------------------ */

/* precision: 0 = the pinned fp32 sequence, 1 = the same sequence in fp64.
 * coords_f64: element type of coords (0 = float, 1 = double); converted to the compute type on load.
 * Other arguments as cdh_histograms (host pointers here).  out is overwritten.  Returns 0, or -1 on
 * an argument the oracle does not accept (it does not validate beyond what it needs). */
int cdh_oracle_histograms(const void *coords, int coords_f64, int n_frames,
                          const int32_t *species_offsets, int n_species, int box_type,
                          const double *box, int n_boxes, double r_max, int n_bins, int precision,
                          int n_threads, uint64_t *out)
{
    if (!coords || !species_offsets || !out || n_frames < 1 || n_species < 1 || n_bins < 1) return -1;
    if (box_type != CDHO_BOX_NONE && (!box || (n_boxes != 1 && n_boxes != n_frames))) return -1;
#ifdef _OPENMP
    if (n_threads > 0) omp_set_num_threads(n_threads);
#else
    (void)n_threads;
#endif
    if (precision == 0)
        return histograms_f32(coords, coords_f64, n_frames, species_offsets, n_species, box_type, box,
                              n_boxes, r_max, n_bins, out);
    return histograms_f64(coords, coords_f64, n_frames, species_offsets, n_species, box_type, box,
                          n_boxes, r_max, n_bins, out);
}

/* Squared minimum-image distance of one pair by the pinned sequence (for the worked examples). */
double cdh_oracle_pair_d2(const double *pi, const double *pj, int box_type, const double *box9,
                          int precision)
{
    return precision == 0 ? single_pair_d2_f32(pi, pj, box_type, box9)
                          : single_pair_d2_f64(pi, pj, box_type, box9);
}

int cdh_oracle_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ------------------------------- g(r) post-processing ------------------------------------- */
/* Radial distribution function from a summed histogram, Eqs. 1-3:
 *   p_kappa = hist[kappa] / N_frames                     (Eq. 2/3: average number of pairs in the bin per frame)
 *   g_kappa = p_kappa / (4 pi (N_pairs / V) r^2 dr)      (Eq. 1 with dr = bin width r_max / n_bins and r taken at
 *                                                         the bin centre (kappa + 1/2) dr -- reading Q15)
 * n_pairs[h] is the number of unique pairs per frame behind histogram h, volume the system volume V.
 * Plain double arithmetic in the order written (no contraction).  Returns 0, or -1 on bad arguments. */
int cdh_oracle_rdf(const uint64_t *hist, int n_hist, int n_bins, double r_max, int n_frames,
                   const double *n_pairs, double volume, double *g)
{
    if (!hist || !n_pairs || !g || n_hist < 1 || n_bins < 1 || n_frames < 1 || !(r_max > 0.0) || !(volume > 0.0))
        return -1;
    const double dr = r_max / (double)n_bins;
    const double four_pi = 4.0 * 3.14159265358979323846;
    for (int h = 0; h < n_hist; ++h) {
        const double density = n_pairs[h] / volume;
        for (int k = 0; k < n_bins; ++k) {
            const double r = ((double)k + 0.5) * dr;
            const double shell = (four_pi * (r * r)) * dr;
            const double p = (double)hist[(size_t)h * (size_t)n_bins + (size_t)k] / (double)n_frames;
            g[(size_t)h * (size_t)n_bins + (size_t)k] = p / (density * shell);
        }
    }
    return 0;
}
