/*
 * oracle/gramsci_oracle.c  --  TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * A plain, slow, obviously-correct CPU implementation (fp64, C99 + OpenMP) of what the
 * GRAMSCI hot path computes: binned counts of 2-, 3- and 4-cliques of the radius graph of a
 * point catalogue, and the parity-decomposed 4-clique counts.  It shares no code with the
 * CUDA path (paper_2607_06604_b200/csrc) and is imported only by tests/, by
 * __graft_entry__.smoke() and by bench.py's cpu_baseline / --impl reference legs.
 *
 * Citations:  P:<n> = /root/reference/PAPER.md line n;  S:8(c) A-k = SURVEY.md section 8(c)
 * reading k (every reading is restated in DESIGN.md).
 *
 * Two independent enumerations live here (S:8(c) "O-def"):
 *   (i)  og_brute_*   : the definition written out -- every index tuple i<j<k(<l), a distance
 *                        test on every pair (O(N^3), O(N^4); tiny N only);
 *   (ii) og_*pcf      : neighbour lists + the paper's walks -- the two-pointer merge-walk of
 *                        P:59-70 for triangles and the three-pointer walk of P:74-87 / Eq. 2 for
 *                        tetrahedra, in the paper's order and notation.
 * (i) pins (ii) (tests/test_oracle_pins.py, with SciPy clique counts, Poisson closed forms,
 * isolated units and the paper's printed configuration counts); (ii) checks the GPU.
 *
 * Parity status: the pixelisation scheme (A-8), the global sign (A-11), the zero weight of
 * bin-achiral configurations and the choice of hub (A-10) are conventions of this build that
 * the paper does not fix -- "parity unpinned" for those four conventions;
 * everything else in the odd channel (antisymmetry under mirroring, recovery of an injected
 * handedness, zero on achiral configurations) is pinned.
 *
 * Build: gcc -O2 -std=c99 -ffp-contract=off -fopenmp -shared -fPIC  (oracle/__init__.py).
 * -ffp-contract=off matters: S:8(c) A-3 fixes d2 = (dx*dx + dy*dy) + dz*dz with every product
 * and sum rounded separately.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define OG_MAXBINS 255

typedef struct {
    int64_t n;
    int nb;
    int periodic;            /* 1 = minimum image with side lengths box[]                      */
    double box[3];
    double r_min, r_max;
    double q[OG_MAXBINS + 1]; /* squared bin edges q_k = e_k*e_k, e_k = r_min + k(r_max-r_min)/nb */
    const double *x;          /* [n,3] caller's points (borrowed)                              */
    double *w;                /* [n] weights (owned copy; all 1.0 when the caller passed NULL)  */
    int weighted;
    /* oriented sorted adjacency lists N+(i) = { j > i : i~j }, S:8(c) A-15, Eq. 1       */
    int64_t *start;           /* [n+1]                                                         */
    int32_t *idx;             /* neighbour label                                               */
    uint8_t *bin;             /* radial-bin byte                                         */
    uint8_t *pix;             /* direction-pixel byte (hub -> spoke, lower -> higher label) */
    /* cell list (only used to find candidate pairs faster; never changes the result)           */
    int nc[3];
    double lo[3], cw[3];
    int64_t *cell_start;      /* [ncell+1] */
    int32_t *cell_pts;        /* [n] point labels grouped by cell, ascending label within a cell */
} og_graph;

/* ------------------------------------------------------------------------------------------ */
/* geometry: S:8(c) A-2, A-3, A-4, A-6                                                           */

static void og_set_edges(og_graph *g)
{
    /* e_k = r_min + (k*(r_max-r_min))/nb, e_0 = r_min, e_nb := r_max ; q_k = e_k*e_k (A-3) */
    for (int k = 0; k <= g->nb; ++k) {
        double e = g->r_min + ((double)k * (g->r_max - g->r_min)) / (double)g->nb;
        if (k == 0) e = g->r_min;
        if (k == g->nb) e = g->r_max;
        g->q[k] = e * e;
    }
}

/* separation vector from point a to point b (minimum image when periodic, A-4) */
static inline void og_sep(const og_graph *g, const double *xa, const double *xb, double d[3])
{
    for (int c = 0; c < 3; ++c) {
        double dx = xb[c] - xa[c];
        if (g->periodic) {
            double L = g->box[c], h = 0.5 * L;
            if (dx > h) dx -= L;
            else if (dx < -h) dx += L;
        }
        d[c] = dx;
    }
}

/* radial bin of a squared distance, or -1 when the pair is not an edge: r_min <= r < r_max (A-2) */
static inline int og_bin_of(const og_graph *g, double d2)
{
    if (!(d2 >= g->q[0] && d2 < g->q[g->nb])) return -1;
    int b = 0;
    for (int k = 1; k < g->nb; ++k)
        if (g->q[k] <= d2) ++b;          /* b = #{k in [1,nb): q_k <= d2} (A-3) */
    return b;
}

static inline double og_d2(const double d[3])
{
    return (d[0] * d[0] + d[1] * d[1]) + d[2] * d[2];     /* (A-3), no FMA contraction */
}

/* direction pixel of a separation vector: 16 z-bands x 16 phi-sectors, equal area (A-8) */
static const double OG_TAN[4] = { 0.0, 0.41421356237309503, 1.0, 2.414213562373095 };

static inline int og_pixel(const double d[3], double d2)
{
    double r = sqrt(d2);
    int iz = 0;
    for (int k = 1; k < 16; ++k)
        if (d[2] >= ((double)k / 8.0 - 1.0) * r) ++iz;    /* iz = #{k in [1,16): dz >= (k/8-1) d} */
    double ax = fabs(d[0]), ay = fabs(d[1]);
    int s = 0;
    for (int k = 1; k <= 3; ++k)
        if (ay >= ax * OG_TAN[k]) ++s;                    /* sub-sector inside the quadrant */
    int iphi;
    if (d[0] >= 0.0) iphi = (d[1] >= 0.0) ? s : 15 - s;   /* quadrants 0 and 3 */
    else             iphi = (d[1] >= 0.0) ? 7 - s : 8 + s; /* quadrants 1 and 2 */
    return 16 * iz + iphi;
}

/* unit vector at the centre of pixel p (A-8): z_c=(iz+1/2)/8-1, phi_c=(iphi+1/2) pi/8 */
void og_pixel_centre(int p, double n[3])
{
    int iz = p >> 4, ip = p & 15;
    double zc = ((double)iz + 0.5) / 8.0 - 1.0;
    double ph = ((double)ip + 0.5) * (3.14159265358979323846 / 8.0);
    double s = sqrt(1.0 - zc * zc);
    n[0] = s * cos(ph);
    n[1] = s * sin(ph);
    n[2] = zc;
}

/* sign of V = (n1 x n2) . n3 with the fixed evaluation order of A-9; 0 when |V| < 1e-9 */
static inline int og_vsign(const double *tab, int p1, int p2, int p3)
{
    const double *a = tab + 3 * p1, *b = tab + 3 * p2, *c = tab + 3 * p3;
    double cx = a[1] * b[2] - a[2] * b[1];
    double cy = a[2] * b[0] - a[0] * b[2];
    double cz = a[0] * b[1] - a[1] * b[0];
    double V = (cx * c[0] + cy * c[1]) + cz * c[2];
    if (fabs(V) < 1e-9) return 0;
    return V > 0.0 ? 1 : -1;
}

/* ------------------------------------------------------------------------------------------ */
/* canonical configurations: S:8(c) A-5, A-7, A-10                                               */

static const int OG_PERM4[24][4] = {
    {0,1,2,3},{0,1,3,2},{0,2,1,3},{0,2,3,1},{0,3,1,2},{0,3,2,1},
    {1,0,2,3},{1,0,3,2},{1,2,0,3},{1,2,3,0},{1,3,0,2},{1,3,2,0},
    {2,0,1,3},{2,0,3,1},{2,1,0,3},{2,1,3,0},{2,3,0,1},{2,3,1,0},
    {3,0,1,2},{3,0,2,1},{3,1,0,2},{3,1,2,0},{3,2,0,1},{3,2,1,0}};

static int og_perm_sign(const int *p)
{
    int inv = 0;
    for (int a = 0; a < 4; ++a)
        for (int b = a + 1; b < 4; ++b)
            if (p[a] > p[b]) ++inv;
    return (inv & 1) ? -1 : 1;
}

/* t = (b01,b02,b03,b12,b13,b23) for vertices 0..3.  Writes the lexicographically minimal
 * re-labelled tuple to c[6] and returns the chirality factor g in {-1,0,+1}:
 *   0  if the minimum is attained by permutations of both parities (achiral at bin resolution),
 *   else the common sign of the attaining permutations (A-10).                                  */
int og_canon4(const int t[6], int c[6])
{
    int m[4][4];
    m[0][1] = m[1][0] = t[0]; m[0][2] = m[2][0] = t[1]; m[0][3] = m[3][0] = t[2];
    m[1][2] = m[2][1] = t[3]; m[1][3] = m[3][1] = t[4]; m[2][3] = m[3][2] = t[5];
    int best[6] = {0,0,0,0,0,0}, have = 0, npos = 0, nneg = 0;
    for (int s = 0; s < 24; ++s) {
        const int *p = OG_PERM4[s];
        int u[6] = { m[p[0]][p[1]], m[p[0]][p[2]], m[p[0]][p[3]],
                     m[p[1]][p[2]], m[p[1]][p[3]], m[p[2]][p[3]] };
        int cmp = 0;
        if (have)
            for (int e = 0; e < 6 && cmp == 0; ++e)
                cmp = (u[e] < best[e]) ? -1 : (u[e] > best[e]) ? 1 : 0;
        if (!have || cmp < 0) {
            memcpy(best, u, sizeof best); have = 1; npos = nneg = 0;
            cmp = 0;
        }
        if (cmp == 0) { if (og_perm_sign(p) > 0) ++npos; else ++nneg; }
    }
    memcpy(c, best, sizeof best);
    if (npos && nneg) return 0;
    return npos ? 1 : -1;
}

static inline int64_t og_index3(int nb, int a, int b, int c) { return ((int64_t)a * nb + b) * nb + c; }

static inline int64_t og_index6(int nb, const int c[6])
{
    int64_t x = 0;
    for (int e = 0; e < 6; ++e) x = x * nb + c[e];
    return x;
}

static inline int64_t og_canon3_index(int nb, int a, int b, int c)
{
    int t;
    if (a > b) { t = a; a = b; b = t; }
    if (b > c) { t = b; b = c; c = t; }
    if (a > b) { t = a; a = b; b = t; }
    return og_index3(nb, a, b, c);         /* sorted triple r1<=r2<=r3 (A-5) */
}

/* number of canonical configurations; optionally list them in lexicographic order
 * (cfg: [n,3] or [n,6] ints, may be NULL).  Pins: 220, 680, 276.          */
int64_t og_num_configs(int npoint, int nb, int32_t *cfg)
{
    int64_t n = 0;
    if (npoint == 3) {
        for (int a = 0; a < nb; ++a) for (int b = a; b < nb; ++b) for (int c = b; c < nb; ++c) {
            if (cfg) { cfg[3*n] = a; cfg[3*n+1] = b; cfg[3*n+2] = c; }
            ++n;
        }
        return n;
    }
    int t[6], c[6];
    for (t[0] = 0; t[0] < nb; ++t[0]) for (t[1] = 0; t[1] < nb; ++t[1])
    for (t[2] = 0; t[2] < nb; ++t[2]) for (t[3] = 0; t[3] < nb; ++t[3])
    for (t[4] = 0; t[4] < nb; ++t[4]) for (t[5] = 0; t[5] < nb; ++t[5]) {
        og_canon4(t, c);
        if (memcmp(t, c, sizeof t) == 0) {
            if (cfg) for (int e = 0; e < 6; ++e) cfg[6*n+e] = t[e];
            ++n;
        }
    }
    return n;
}

/* ------------------------------------------------------------------------------------------ */
/* graph construction: P:39-47 (S:8(c) O-def step 1).  use_cells = 0: all N(N-1)/2 pairs.         */

static void og_build_cells(og_graph *g)
{
    const int64_t n = g->n;
    for (int c = 0; c < 3; ++c) {
        double lo, hi;
        if (g->periodic) { lo = 0.0; hi = g->box[c]; }
        else {
            lo = hi = n ? g->x[c] : 0.0;
            for (int64_t i = 0; i < n; ++i) {
                double v = g->x[3*i+c];
                if (v < lo) lo = v;
                if (v > hi) hi = v;
            }
        }
        double ext = hi - lo;
        int nc = (int)floor(ext / g->r_max);
        if (nc < 1) nc = 1;
        if (nc > 256) nc = 256;
        g->nc[c] = nc; g->lo[c] = lo; g->cw[c] = ext / nc;
        if (!(g->cw[c] > 0.0)) g->cw[c] = 1.0;
    }
    int64_t ncell = (int64_t)g->nc[0] * g->nc[1] * g->nc[2];
    g->cell_start = (int64_t *)calloc((size_t)ncell + 1, sizeof(int64_t));
    g->cell_pts = (int32_t *)malloc((size_t)(n ? n : 1) * sizeof(int32_t));
    int64_t *cid = (int64_t *)malloc((size_t)(n ? n : 1) * sizeof(int64_t));
    for (int64_t i = 0; i < n; ++i) {
        int64_t id = 0;
        for (int c = 2; c >= 0; --c) {
            int k = (int)floor((g->x[3*i+c] - g->lo[c]) / g->cw[c]);
            if (k < 0) k = 0;
            if (k >= g->nc[c]) k = g->nc[c] - 1;
            id = id * g->nc[c] + k;
        }
        cid[i] = id;
        g->cell_start[id + 1]++;
    }
    for (int64_t c = 0; c < ncell; ++c) g->cell_start[c + 1] += g->cell_start[c];
    int64_t *fill = (int64_t *)malloc((size_t)ncell * sizeof(int64_t));
    memcpy(fill, g->cell_start, (size_t)ncell * sizeof(int64_t));
    for (int64_t i = 0; i < n; ++i) g->cell_pts[fill[cid[i]]++] = (int32_t)i;   /* ascending label */
    free(fill); free(cid);
}

typedef struct { int32_t j; uint8_t b, p; } og_ent;

static int og_ent_cmp(const void *a, const void *b)
{
    int32_t x = ((const og_ent *)a)->j, y = ((const og_ent *)b)->j;
    return (x > y) - (x < y);
}

/* all j != i with an edge to i and (j > i or !oriented); returns count, appends to *buf */
static int64_t og_row_of(const og_graph *g, int64_t i, int use_cells, int oriented,
                         og_ent **buf, int64_t *cap)
{
    int64_t m = 0;
    const double *xi = g->x + 3*i;
#define OG_TRY(J) do { int64_t j_ = (J); if (j_ != i && (!oriented || j_ > i)) {                    \
        double d[3]; const double *xj = g->x + 3*j_;                                                \
        /* direction lower label -> higher label (hub -> spoke) */                                  \
        if (j_ > i) og_sep(g, xi, xj, d); else og_sep(g, xj, xi, d);                                \
        double d2 = og_d2(d); int b_ = og_bin_of(g, d2);                                            \
        if (b_ >= 0) { if (m == *cap) { *cap = *cap ? 2 * *cap : 256;                               \
                                        *buf = (og_ent *)realloc(*buf, (size_t)*cap * sizeof(og_ent)); } \
            (*buf)[m].j = (int32_t)j_; (*buf)[m].b = (uint8_t)b_; (*buf)[m].p = (uint8_t)og_pixel(d, d2); ++m; } } } while (0)
    if (!use_cells) {
        for (int64_t j = 0; j < g->n; ++j) OG_TRY(j);
    } else {
        int ci[3];
        for (int c = 0; c < 3; ++c) {
            int k = (int)floor((xi[c] - g->lo[c]) / g->cw[c]);
            if (k < 0) k = 0;
            if (k >= g->nc[c]) k = g->nc[c] - 1;
            ci[c] = k;
        }
        /* distinct neighbouring cells (periodic wrap may alias offsets when nc < 3) */
        int64_t seen[27]; int ns = 0;
        for (int dz = -1; dz <= 1; ++dz) for (int dy = -1; dy <= 1; ++dy) for (int dx = -1; dx <= 1; ++dx) {
            int o[3] = { ci[0] + dx, ci[1] + dy, ci[2] + dz }, ok = 1;
            for (int c = 0; c < 3; ++c) {
                if (g->periodic) o[c] = ((o[c] % g->nc[c]) + g->nc[c]) % g->nc[c];
                else if (o[c] < 0 || o[c] >= g->nc[c]) ok = 0;
            }
            if (!ok) continue;
            int64_t id = ((int64_t)o[2] * g->nc[1] + o[1]) * g->nc[0] + o[0];
            int dup = 0;
            for (int s = 0; s < ns; ++s) if (seen[s] == id) dup = 1;
            if (dup) continue;
            seen[ns++] = id;
            for (int64_t s = g->cell_start[id]; s < g->cell_start[id + 1]; ++s) OG_TRY(g->cell_pts[s]);
        }
    }
#undef OG_TRY
    qsort(*buf, (size_t)m, sizeof(og_ent), og_ent_cmp);     /* Eq. 1: j1 < j2 < ... */
    return m;
}

void og_free(og_graph *g)
{
    if (!g) return;
    free(g->w); free(g->start); free(g->idx); free(g->bin); free(g->pix);
    free(g->cell_start); free(g->cell_pts); free(g);
}

/* lists = 0: only parameters + cell list (for the *_direct functions); lists = 1: full graph */
og_graph *og_build(const double *pts, const double *w, int64_t n, const double *box,
                   double r_min, double r_max, int nb, int use_cells, int lists)
{
    if (n < 0 || nb < 1 || nb > OG_MAXBINS || !(r_max > r_min) || r_min < 0.0) return NULL;
    og_graph *g = (og_graph *)calloc(1, sizeof(og_graph));
    g->n = n; g->nb = nb; g->r_min = r_min; g->r_max = r_max; g->x = pts;
    g->periodic = (box && box[0] > 0.0 && box[1] > 0.0 && box[2] > 0.0);
    if (g->periodic) {
        for (int c = 0; c < 3; ++c) {
            g->box[c] = box[c];
            if (!(r_max < 0.5 * box[c])) { free(g); return NULL; }     /* A-4 */
        }
    }
    og_set_edges(g);
    g->w = (double *)malloc((size_t)(n ? n : 1) * sizeof(double));
    g->weighted = (w != NULL);
    for (int64_t i = 0; i < n; ++i) g->w[i] = w ? w[i] : 1.0;
    og_build_cells(g);
    if (!lists) return g;

    g->start = (int64_t *)calloc((size_t)n + 1, sizeof(int64_t));
    og_ent **rows = (og_ent **)calloc((size_t)(n ? n : 1), sizeof(og_ent *));
#pragma omp parallel
    {
        og_ent *buf = NULL; int64_t cap = 0;
#pragma omp for schedule(dynamic, 64)
        for (int64_t i = 0; i < n; ++i) {
            int64_t m = og_row_of(g, i, use_cells, 1, &buf, &cap);
            g->start[i + 1] = m;
            rows[i] = (og_ent *)malloc((size_t)(m ? m : 1) * sizeof(og_ent));
            memcpy(rows[i], buf, (size_t)m * sizeof(og_ent));
        }
        free(buf);
    }
    for (int64_t i = 0; i < n; ++i) g->start[i + 1] += g->start[i];
    int64_t E = g->start[n];
    g->idx = (int32_t *)malloc((size_t)(E ? E : 1) * sizeof(int32_t));
    g->bin = (uint8_t *)malloc((size_t)(E ? E : 1));
    g->pix = (uint8_t *)malloc((size_t)(E ? E : 1));
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) {
        int64_t s = g->start[i], m = g->start[i + 1] - s;
        for (int64_t k = 0; k < m; ++k) {
            g->idx[s + k] = rows[i][k].j; g->bin[s + k] = rows[i][k].b; g->pix[s + k] = rows[i][k].p;
        }
        free(rows[i]);
    }
    free(rows);
    return g;
}

int64_t og_num_edges(const og_graph *g) { return g->start ? g->start[g->n] : -1; }

/* copy the CSR out (for graph-level parity against the GPU build) */
void og_export(const og_graph *g, int64_t *start, int32_t *idx, uint8_t *bin, uint8_t *pix)
{
    memcpy(start, g->start, (size_t)(g->n + 1) * sizeof(int64_t));
    int64_t E = g->start[g->n];
    if (idx) memcpy(idx, g->idx, (size_t)E * sizeof(int32_t));
    if (bin) memcpy(bin, g->bin, (size_t)E);
    if (pix) memcpy(pix, g->pix, (size_t)E);
}

/* ------------------------------------------------------------------------------------------ */
/* hub filter shared by every query: hub i is processed iff                                       */
/*   hub_begin <= i < hub_end  and  (i - hub_begin) % hub_stride == 0.                            */
/* A "hub" is the smallest-label vertex of the tuple (A-1: each tuple once, i<j<k<l).            */

static inline int og_hub_ok(int64_t i, int64_t hb, int64_t he, int64_t hs)
{
    return i >= hb && i < he && ((i - hb) % (hs > 0 ? hs : 1)) == 0;
}

static int og_nthreads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
int og_threads(void) { return og_nthreads(); }

/* ------------------------------------------------------------------------------------------ */
/* 2pCF sweep: P:118 (O-def step 2).  cnt [nb] int64, wsum [nb] double (either may be NULL)       */

void og_2pcf(const og_graph *g, int64_t *cnt, double *wsum)
{
    int nb = g->nb;
    long double *acc = (long double *)calloc((size_t)nb, sizeof(long double));
    int64_t *c = (int64_t *)calloc((size_t)nb, sizeof(int64_t));
    for (int64_t i = 0; i < g->n; ++i)
        for (int64_t s = g->start[i]; s < g->start[i + 1]; ++s) {
            c[g->bin[s]] += 1;
            acc[g->bin[s]] += (long double)g->w[i] * (long double)g->w[g->idx[s]];
        }
    for (int b = 0; b < nb; ++b) { if (cnt) cnt[b] = c[b]; if (wsum) wsum[b] = (double)acc[b]; }
    free(acc); free(c);
}

/* ------------------------------------------------------------------------------------------ */
/* 3pCF: hub-and-spoke loop with the two-pointer merge-walk, P:51 + P:59-70.                      */
/* cnt [nb^3] int64, wsum [nb^3] double, dense, populated at sorted triples only (A-5).           */

void og_3pcf(const og_graph *g, int64_t *cnt, double *wsum,
             int64_t hub_begin, int64_t hub_end, int64_t hub_stride)
{
    const int nb = g->nb;
    const int64_t nh = (int64_t)nb * nb * nb;
    const int nt = og_nthreads();
    int64_t *C = (int64_t *)calloc((size_t)nh * nt, sizeof(int64_t));
    long double *W = (long double *)calloc((size_t)nh * nt, sizeof(long double));
#pragma omp parallel
    {
#ifdef _OPENMP
        int t = omp_get_thread_num();
#else
        int t = 0;
#endif
        int64_t *c = C + (size_t)nh * t;
        long double *wacc = W + (size_t)nh * t;
#pragma omp for schedule(dynamic, 16)
        for (int64_t i = 0; i < g->n; ++i) {                     /* hub i */
            if (!og_hub_ok(i, hub_begin, hub_end, hub_stride)) continue;
            const int64_t is = g->start[i], ie = g->start[i + 1];
            for (int64_t sj = is; sj < ie; ++sj) {               /* spoke j in N(i) */
                const int32_t j = g->idx[sj];
                int64_t a = sj + 1;                              /* a: hub tail, entry after j */
                int64_t b = g->start[j];                         /* b: N(j) from its beginning */
                const int64_t be = g->start[j + 1];
                while (a < ie && b < be) {
                    int32_t ha = g->idx[a], hb = g->idx[b];
                    if (ha == hb) {                              /* triangle (i,j,k) found */
                        int64_t x = og_canon3_index(nb, g->bin[sj], g->bin[a], g->bin[b]);
                        c[x] += 1;
                        wacc[x] += (long double)g->w[i] * (long double)g->w[j] * (long double)g->w[ha];
                        ++a; ++b;
                    } else if (ha < hb) ++a;
                    else ++b;
                }
            }
        }
    }
    for (int64_t x = 0; x < nh; ++x) {
        int64_t s = 0; long double ws = 0.0L;
        for (int t = 0; t < nt; ++t) { s += C[(size_t)nh * t + x]; ws += W[(size_t)nh * t + x]; }
        if (cnt) cnt[x] = s;
        if (wsum) wsum[x] = (double)ws;
    }
    free(C); free(W);
}

/* ------------------------------------------------------------------------------------------ */
/* 4pCF and parity 4pCF: two-pointer walk for j2, three-pointer walk (Eq. 2) for j3.     */
/* Outputs dense [nb^6] (order b12,b13,b14,b23,b24,b34), populated at canonical tuples (A-7).     */
/* parity = 0: odd_* ignored.  odd_cnt is int64 (signed).                                         */

void og_4pcf(const og_graph *g, int parity, int64_t *even_cnt, double *even_w,
             int64_t *odd_cnt, double *odd_w,
             int64_t hub_begin, int64_t hub_end, int64_t hub_stride)
{
    const int nb = g->nb;
    int64_t nh = 1;
    for (int e = 0; e < 6; ++e) nh *= nb;
    /* raw 6-tuple -> (compact canonical id, chirality factor g) lookup, built from og_canon4 */
    int32_t *cid = (int32_t *)malloc((size_t)nh * sizeof(int32_t));
    int8_t *chi = (int8_t *)malloc((size_t)nh);
    int64_t *dense_of = (int64_t *)malloc((size_t)nh * sizeof(int64_t));
    int64_t ncfg = 0;
    {
        int t[6], c[6];
        for (int64_t x = 0; x < nh; ++x) {            /* first pass: number the canonical tuples */
            int64_t r = x;
            for (int e = 5; e >= 0; --e) { t[e] = (int)(r % nb); r /= nb; }
            og_canon4(t, c);
            if (og_index6(nb, c) == x) { cid[x] = (int32_t)ncfg; dense_of[ncfg] = x; ++ncfg; }
        }
        for (int64_t x = 0; x < nh; ++x) {
            int64_t r = x;
            for (int e = 5; e >= 0; --e) { t[e] = (int)(r % nb); r /= nb; }
            chi[x] = (int8_t)og_canon4(t, c);
            cid[x] = cid[og_index6(nb, c)];
        }
    }
    double tab[256 * 3];
    for (int p = 0; p < 256; ++p) og_pixel_centre(p, tab + 3 * p);

    const int nt = og_nthreads();
    int64_t *CE = (int64_t *)calloc((size_t)ncfg * nt, sizeof(int64_t));
    int64_t *CO = (int64_t *)calloc((size_t)ncfg * nt, sizeof(int64_t));
    long double *WE = (long double *)calloc((size_t)ncfg * nt, sizeof(long double));
    long double *WO = (long double *)calloc((size_t)ncfg * nt, sizeof(long double));
#pragma omp parallel
    {
#ifdef _OPENMP
        int th = omp_get_thread_num();
#else
        int th = 0;
#endif
        int64_t *ce = CE + (size_t)ncfg * th, *co = CO + (size_t)ncfg * th;
        long double *we = WE + (size_t)ncfg * th, *wo = WO + (size_t)ncfg * th;
#pragma omp for schedule(dynamic, 4)
        for (int64_t i = 0; i < g->n; ++i) {                       /* hub i */
            if (!og_hub_ok(i, hub_begin, hub_end, hub_stride)) continue;
            const int64_t is = g->start[i], ie = g->start[i + 1];
            for (int64_t s1 = is; s1 < ie; ++s1) {                 /* first spoke j1 */
                const int32_t j1 = g->idx[s1];
                int64_t a = s1 + 1, b = g->start[j1];
                const int64_t b1e = g->start[j1 + 1];
                while (a < ie && b < b1e) {                        /* k2 walk: find j2 */
                    int32_t ha = g->idx[a], hb = g->idx[b];
                    if (ha < hb) { ++a; continue; }
                    if (hb < ha) { ++b; continue; }
                    const int32_t j2 = ha;                         /* second spoke located */
                    int64_t al = a + 1;                            /* alpha: hub tail beyond j2 */
                    int64_t be = b + 1;                            /* beta : N(j1) just after j2 */
                    int64_t ga = g->start[j2];                     /* gamma: N(j2); oriented lists hold
                                                                      only entries > j2 already */
                    const int64_t g2e = g->start[j2 + 1];
                    while (al < ie && be < b1e && ga < g2e) {
                        int32_t h_al = g->idx[al], h_be = g->idx[be], h_ga = g->idx[ga];
                        if (h_al == h_be && h_be == h_ga) {        /* tetrahedron (i,j1,j2,j3) */
                            int t[6] = { g->bin[s1], g->bin[a], g->bin[al],      /* b_ij1 b_ij2 b_ij3 */
                                         g->bin[b], g->bin[be], g->bin[ga] };    /* b_j1j2 b_j1j3 b_j2j3 */
                            int64_t x = og_index6(nb, t);
                            int32_t cc = cid[x];
                            long double ww = (long double)g->w[i] * (long double)g->w[j1] *
                                             (long double)g->w[j2] * (long double)g->w[h_al];
                            ce[cc] += 1; we[cc] += ww;
                            if (parity) {
                                /* Eq. 3 on pixel centres, hub = smallest label, spokes ascending (A-9, A-10) */
                                int sg = chi[x] * og_vsign(tab, g->pix[s1], g->pix[a], g->pix[al]);
                                co[cc] += sg; wo[cc] += (long double)sg * ww;
                            }
                            ++al; ++be; ++ga;
                        } else {                                   /* Eq. 2: advance every pointer at the minimum */
                            int adv_al = (h_al <= h_be && h_al <= h_ga);
                            int adv_be = (h_be <= h_al && h_be <= h_ga);
                            int adv_ga = (h_ga <= h_al && h_ga <= h_be);
                            al += adv_al; be += adv_be; ga += adv_ga;
                        }
                    }
                    ++a; ++b;
                }
            }
        }
    }
    if (even_cnt) memset(even_cnt, 0, (size_t)nh * sizeof(int64_t));
    if (even_w) memset(even_w, 0, (size_t)nh * sizeof(double));
    if (parity && odd_cnt) memset(odd_cnt, 0, (size_t)nh * sizeof(int64_t));
    if (parity && odd_w) memset(odd_w, 0, (size_t)nh * sizeof(double));
    for (int64_t k = 0; k < ncfg; ++k) {
        int64_t se = 0, so = 0; long double te = 0.0L, to = 0.0L;
        for (int t = 0; t < nt; ++t) {
            se += CE[(size_t)ncfg * t + k]; so += CO[(size_t)ncfg * t + k];
            te += WE[(size_t)ncfg * t + k]; to += WO[(size_t)ncfg * t + k];
        }
        int64_t x = dense_of[k];
        if (even_cnt) even_cnt[x] = se;
        if (even_w) even_w[x] = (double)te;
        if (parity && odd_cnt) odd_cnt[x] = so;
        if (parity && odd_w) odd_w[x] = (double)to;
    }
    free(CE); free(CO); free(WE); free(WO); free(cid); free(chi); free(dense_of);
}

/* ------------------------------------------------------------------------------------------ */
/* (i) brute force: the definition written out on index tuples; no lists, no cells, no walks.      */

static inline int og_pair(const og_graph *g, int64_t a, int64_t b, int *pixel)
{   /* a < b ; returns bin or -1 */
    double d[3];
    og_sep(g, g->x + 3*a, g->x + 3*b, d);
    double d2 = og_d2(d);
    int bb = og_bin_of(g, d2);
    if (bb >= 0 && pixel) *pixel = og_pixel(d, d2);
    return bb;
}

void og_brute_2pcf(const og_graph *g, int64_t *cnt, double *wsum)
{
    for (int b = 0; b < g->nb; ++b) { if (cnt) cnt[b] = 0; if (wsum) wsum[b] = 0.0; }
    for (int64_t i = 0; i < g->n; ++i) for (int64_t j = i + 1; j < g->n; ++j) {
        int b = og_pair(g, i, j, NULL);
        if (b < 0) continue;
        if (cnt) cnt[b] += 1;
        if (wsum) wsum[b] += g->w[i] * g->w[j];
    }
}

void og_brute_3pcf(const og_graph *g, int64_t *cnt, double *wsum)
{
    const int nb = g->nb; const int64_t nh = (int64_t)nb * nb * nb;
    if (cnt) memset(cnt, 0, (size_t)nh * sizeof(int64_t));
    if (wsum) memset(wsum, 0, (size_t)nh * sizeof(double));
    for (int64_t i = 0; i < g->n; ++i) for (int64_t j = i + 1; j < g->n; ++j) {
        int bij = og_pair(g, i, j, NULL);
        if (bij < 0) continue;
        for (int64_t k = j + 1; k < g->n; ++k) {
            int bik = og_pair(g, i, k, NULL); if (bik < 0) continue;
            int bjk = og_pair(g, j, k, NULL); if (bjk < 0) continue;
            int64_t x = og_canon3_index(nb, bij, bik, bjk);
            if (cnt) cnt[x] += 1;
            if (wsum) wsum[x] += g->w[i] * g->w[j] * g->w[k];
        }
    }
}

void og_brute_4pcf(const og_graph *g, int parity, int64_t *even_cnt, double *even_w,
                   int64_t *odd_cnt, double *odd_w)
{
    const int nb = g->nb; int64_t nh = 1;
    for (int e = 0; e < 6; ++e) nh *= nb;
    if (even_cnt) memset(even_cnt, 0, (size_t)nh * sizeof(int64_t));
    if (even_w) memset(even_w, 0, (size_t)nh * sizeof(double));
    if (parity && odd_cnt) memset(odd_cnt, 0, (size_t)nh * sizeof(int64_t));
    if (parity && odd_w) memset(odd_w, 0, (size_t)nh * sizeof(double));
    double tab[256 * 3];
    for (int p = 0; p < 256; ++p) og_pixel_centre(p, tab + 3 * p);
    for (int64_t i = 0; i < g->n; ++i) for (int64_t j = i + 1; j < g->n; ++j) {
        int p1 = 0, p2 = 0, p3 = 0;
        int b01 = og_pair(g, i, j, &p1); if (b01 < 0) continue;
        for (int64_t k = j + 1; k < g->n; ++k) {
            int b02 = og_pair(g, i, k, &p2); if (b02 < 0) continue;
            int b12 = og_pair(g, j, k, NULL); if (b12 < 0) continue;
            for (int64_t l = k + 1; l < g->n; ++l) {
                int b03 = og_pair(g, i, l, &p3); if (b03 < 0) continue;
                int b13 = og_pair(g, j, l, NULL); if (b13 < 0) continue;
                int b23 = og_pair(g, k, l, NULL); if (b23 < 0) continue;
                int t[6] = { b01, b02, b03, b12, b13, b23 }, c[6];
                int chi = og_canon4(t, c);
                int64_t x = og_index6(nb, c);
                double ww = g->w[i] * g->w[j] * g->w[k] * g->w[l];
                if (even_cnt) even_cnt[x] += 1;
                if (even_w) even_w[x] += ww;
                if (parity) {
                    int sg = chi * og_vsign(tab, p1, p2, p3);
                    if (odd_cnt) odd_cnt[x] += sg;
                    if (odd_w) odd_w[x] += sg * ww;
                }
            }
        }
    }
}

/* ------------------------------------------------------------------------------------------ */
/* sampled hubs on graphs too large to hold: the same 3pCF walk, but the rows of the hub and of   */
/* its spokes are found on demand from the cell list (g built with lists = 0).                     */

void og_3pcf_direct(const og_graph *g, const int64_t *hubs, int64_t nhubs, int64_t *cnt, double *wsum)
{
    const int nb = g->nb; const int64_t nh = (int64_t)nb * nb * nb;
    const int nt = og_nthreads();
    int64_t *C = (int64_t *)calloc((size_t)nh * nt, sizeof(int64_t));
    long double *W = (long double *)calloc((size_t)nh * nt, sizeof(long double));
    for (int64_t h = 0; h < nhubs; ++h) {
        const int64_t i = hubs[h];
        og_ent *ri = NULL; int64_t capi = 0;
        const int64_t mi = og_row_of(g, i, 1, 1, &ri, &capi);
#pragma omp parallel
        {
#ifdef _OPENMP
            int t = omp_get_thread_num();
#else
            int t = 0;
#endif
            og_ent *rj = NULL; int64_t capj = 0;
#pragma omp for schedule(dynamic, 8)
            for (int64_t sj = 0; sj < mi; ++sj) {
                const int32_t j = ri[sj].j;
                const int64_t mj = og_row_of(g, j, 1, 1, &rj, &capj);
                int64_t a = sj + 1, b = 0;
                while (a < mi && b < mj) {
                    if (ri[a].j == rj[b].j) {
                        int64_t x = og_canon3_index(nb, ri[sj].b, ri[a].b, rj[b].b);
                        C[(size_t)nh * t + x] += 1;
                        W[(size_t)nh * t + x] += (long double)g->w[i] * (long double)g->w[j] * (long double)g->w[ri[a].j];
                        ++a; ++b;
                    } else if (ri[a].j < rj[b].j) ++a;
                    else ++b;
                }
            }
            free(rj);
        }
        free(ri);
    }
    for (int64_t x = 0; x < nh; ++x) {
        int64_t s = 0; long double ws = 0.0L;
        for (int t = 0; t < nt; ++t) { s += C[(size_t)nh * t + x]; ws += W[(size_t)nh * t + x]; }
        if (cnt) cnt[x] = s;
        if (wsum) wsum[x] = (double)ws;
    }
    free(C); free(W);
}

/* degree (full, both directions) and oriented degree of selected points, from the cell list */
void og_degrees_direct(const og_graph *g, const int64_t *pts, int64_t npts, int64_t *full_deg, int64_t *plus_deg)
{
#pragma omp parallel
    {
        og_ent *r = NULL; int64_t cap = 0;
#pragma omp for schedule(dynamic, 8)
        for (int64_t h = 0; h < npts; ++h) {
            if (full_deg) full_deg[h] = og_row_of(g, pts[h], 1, 0, &r, &cap);
            if (plus_deg) plus_deg[h] = og_row_of(g, pts[h], 1, 1, &r, &cap);
        }
        free(r);
    }
}

/* ------------------------------------------------------------------------------------------ */
/* disconnected 4pCF, Eq. 4: zeta_disc[c] = xi(c12)xi(c34)+xi(c13)xi(c24)+xi(c14)xi(c23)   */
/* evaluated on every dense index (it is S4-invariant).  xi [nb] -> out [nb^6].             */

void og_zeta_disc(int nb, const double *xi, double *out)
{
    int64_t nh = 1;
    for (int e = 0; e < 6; ++e) nh *= nb;
    for (int64_t x = 0; x < nh; ++x) {
        int t[6]; int64_t r = x;
        for (int e = 5; e >= 0; --e) { t[e] = (int)(r % nb); r /= nb; }
        /* t = (b12,b13,b14,b23,b24,b34) */
        out[x] = xi[t[0]] * xi[t[5]] + xi[t[1]] * xi[t[4]] + xi[t[2]] * xi[t[3]];
    }
}
