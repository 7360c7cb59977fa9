/*
 * nhp_oracle.c -- TEST INFRASTRUCTURE ONLY.
 *
 * Plain, slow, sequential CPU statement of what the hot path of
 * "Nonholonomic Motion Planning as Efficient as Piano Mover's" (arXiv 2306.01301,
 * /root/reference/PAPER.md) computes.  Only tests/, __graft_entry__.smoke() and the
 * cpu_baseline / --impl reference legs of bench.py may load this library.  It shares no
 * code, header, table or constant generator with the CUDA path under
 * paper_2306_01301_b200/csrc/ and neither side includes the other.
 *
 * Every function cites the passage of PAPER.md (line + section/equation) it follows;
 * "DESIGN R<k>" refers to the numbered readings in /root/repo/DESIGN.md where the paper is
 * silent, garbled or ambiguous.
 *
 * Parity pins (tests/test_oracle_*.py, all `-m "not gpu"`):
 *   tables ........ Psi2=Psi0, Psi3=Psi1, snap error <= 1/4 and <= 1/2, plane step <= 1
 *                   (Lemma 4/5 l.779-785), curve maps are bijections (l.224,269,302)
 *   edge maps ..... LB o LF = id etc., edge(p) = curve-map(step+1)             (l.306, l.320)
 *   sweeps ........ closed form on one curve, fix-point == Star Dijkstra == Compact Dijkstra,
 *                   layered brute-force DP on tiny grids, 26-neighbour Piano-mover relaxation (l.88);
 *                   free-space fix-point against the Dubins / Reeds-Shepp closed forms within the bounds of
 *                   Theorems 1, 6, 7 (l.104, 809, 815): tests/test_oracle_reeds_shepp.py, tests/closed_forms.py
 *   graph sizes ... k_V / k_E of Table 1 (l.427) counted on the Dijkstra itself (tests/test_oracle_tables.py)
 *   render ........ brute force vs exact box dilation at axis angles; run renderer vs brute force
 *   back-track .... plan is a valid chain of curve segments whose cost sums to the reported cost
 *   lane penalty .. (DESIGN R28, our definition) factor 16 = identity bit for bit, aligned heading unpenalised, opposite heading
 *                   exactly x pen/16, symmetric and monotone in the angle and in pen, saturation; in free space a straight drive
 *                   with the lane costs what it costs without the penalty and against it exactly pen/16 times that
 *                   (tests/test_oracle_lane.py)
 *   orc_render_*'s footprint rasterisation rule (DESIGN R15) is OUR definition: "parity
 *   unpinned" against the paper, which gives no rule.
 *
 * Conventions:
 *   volume index  idx = (Theta*N + j)*N + i,  i = x fastest
 *   maneuver ids in cycle order: 0 LF, 1 SF, 2 RB, 3 RF, 4 SB, 5 LB
 *   costs: uint32, unit 1/2^cost_one_log2 cell; INF = 0xFFFFFFFF; a (+) b saturates to INF
 *   as soon as the exact sum reaches LIMIT = 2^30 (DESIGN R18).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_PI 3.14159265358979323846
#define ORC_INF 0xFFFFFFFFu
#define ORC_LIMIT (1ull << 30)
#define ORC_FLAG_FORWARD_ONLY 1

enum { M_LF = 0, M_SF = 1, M_RB = 2, M_RF = 3, M_SB = 4, M_LB = 5 };

typedef struct {
    int32_t log2_n, log2_nt;
    double R;               /* minimum turn radius in cells */
    uint32_t ct[6];         /* transition-in cost per maneuver, cost units */
    uint32_t dir_mult[6];   /* Q8.8 length multiplier per maneuver (256 = x1) */
    int32_t cost_one_log2;
    int32_t flags;
} orc_params;

typedef struct {
    const uint8_t *mask;    /* mh rows x mw cols; column p along the vehicle's length axis u */
    int32_t mw, mh;
    double ou, ov;          /* mask pixel (p,q) owns the unit square centred (p-ou, q-ov) */
} orc_footprint;

typedef struct {
    int32_t i, j, theta, m; /* m = maneuver that arrives at this waypoint from the next one; -1 at the start */
} orc_waypoint;

typedef struct orc_ctx {
    orc_params p;
    int n, nt, mx, mt;
    int32_t *beta;     /* [nt]   beta(Theta)                      eq (13)-(17) */
    uint8_t *psi2;     /* [nt]   2*Psi(Theta) in {0,1}            eq (13) */
    uint8_t *I;        /* [nt]   octant class                     eq (19) */
    int8_t *J;         /* [nt]   forward sign                     eq (24) */
    double *K;         /* [nt]   tan or cot                       eq (20) */
    int32_t *B;        /* [nt][n] B(y',Theta) = round(y' K)        l.284 */
    uint32_t *len_q;   /* [6][nt] fixed-point edge length         l.334 */
    int32_t *cosq, *sinq; /* [nt] round(2^14 cos/sin theta)        DESIGN R15 */
    int threads;
} orc_ctx;

/* ------------------------------------------------------------------------------------------
 * Trigonometry with exact symmetries.  theta(Theta) = 2 pi Theta / N_theta.
 * The argument is reduced to the first octant with integer arithmetic so that
 * sin(theta+pi) = -sin(theta), sin(pi-theta) = sin(theta) and sin(pi/4) = cos(pi/4) hold
 * bit-for-bit; the identities Psi2=Psi0, Psi3=Psi1 of PAPER.md:247 need exactly that.
 * ---------------------------------------------------------------------------------------- */
static double sin_turn(int k, int nt)
{
    int half = nt / 2, q = nt / 4;
    double sg = 1.0, s;
    k &= nt - 1;
    if (k >= half) { k -= half; sg = -1.0; }
    if (k > q) k = half - k;
    if (k == 0) s = 0.0;
    else if (k == q) s = 1.0;
    else if (2 * k <= q) s = sin(2.0 * ORC_PI * (double)k / (double)nt);
    else s = cos(2.0 * ORC_PI * (double)(q - k) / (double)nt);
    return sg * s;
}
static double cos_turn(int k, int nt) { return sin_turn(k + nt / 4, nt); }

/* zeta(x) = round(2x)/2; round = half away from zero (DESIGN R4). */
static double zeta(double x) { return round(2.0 * x) / 2.0; }

static int64_t floordiv(int64_t a, int64_t b) /* b > 0 */
{
    int64_t q = a / b;
    if ((a % b) != 0 && a < 0) q -= 1;
    return q;
}

/* Saturating cost addition, DESIGN R18. */
static uint32_t cadd(uint32_t a, uint32_t b)
{
    if (a == ORC_INF || b == ORC_INF) return ORC_INF;
    uint64_t s = (uint64_t)a + (uint64_t)b;
    return s >= ORC_LIMIT ? ORC_INF : (uint32_t)s;
}

void orc_destroy(orc_ctx *c)
{
    if (!c) return;
    free(c->beta); free(c->psi2); free(c->I); free(c->J); free(c->K); free(c->B);
    free(c->len_q); free(c->cosq); free(c->sinq); free(c);
}

/* Table build: PAPER.md:226-302 (section V.C), l.334 (edge lengths).  Returns NULL on bad
 * parameters; *err: 1 bad arg, 2 N_theta < 2 pi R (DESIGN R23), 3 weights too large. */
orc_ctx *orc_create(const orc_params *p, int *err)
{
    int e = 0;
    if (!p || p->log2_n < 3 || p->log2_n > 12 || p->log2_nt < 3 || p->log2_nt > 12 ||
        !(p->R >= 1.0) || p->cost_one_log2 < 0 || p->cost_one_log2 > 16) e = 1;
    if (!e && (double)(1 << p->log2_nt) < 2.0 * ORC_PI * p->R) e = 2;
    if (e) { if (err) *err = e; return NULL; }
    orc_ctx *c = (orc_ctx *)calloc(1, sizeof(orc_ctx));
    c->p = *p;
    c->n = 1 << p->log2_n; c->nt = 1 << p->log2_nt; c->mx = c->n - 1; c->mt = c->nt - 1;
    c->threads = 1;
    int n = c->n, nt = c->nt;
    c->beta = (int32_t *)malloc(sizeof(int32_t) * nt);
    c->psi2 = (uint8_t *)malloc(nt);
    c->I = (uint8_t *)malloc(nt);
    c->J = (int8_t *)malloc(nt);
    c->K = (double *)malloc(sizeof(double) * nt);
    c->B = (int32_t *)malloc(sizeof(int32_t) * (size_t)nt * n);
    c->len_q = (uint32_t *)malloc(sizeof(uint32_t) * 6 * nt);
    c->cosq = (int32_t *)malloc(sizeof(int32_t) * nt);
    c->sinq = (int32_t *)malloc(sizeof(int32_t) * nt);
    double one = (double)(1u << p->cost_one_log2);
    for (int t = 0; t < nt; t++) {
        double s = sin_turn(t, nt), co = cos_turn(t, nt);
        /* alpha, zeta, beta = floor(zeta(alpha)) (DESIGN R3), Psi: PAPER.md:233-240 */
        double z = zeta(p->R * s);
        double b = floor(z);
        c->beta[t] = (int32_t)b;
        c->psi2[t] = (uint8_t)(int)(2.0 * (z - b));
        /* eq (19): I = 0 iff |tan| <= 1, decided on the integer octant (DESIGN R5) */
        int o = t & (nt / 2 - 1);
        int I = (o <= nt / 8 || o >= 3 * nt / 8) ? 0 : 1;
        c->I[t] = (uint8_t)I;
        /* eq (20), eq (24) */
        c->K[t] = I == 0 ? s / co : co / s;
        double f = I == 0 ? co : s;
        c->J[t] = (int8_t)(f > 0 ? 1 : -1);
        for (int y = 0; y < n; y++) c->B[(size_t)t * n + y] = (int32_t)round((double)y * c->K[t]);
        /* edge lengths; fixed point per DESIGN R18 */
        double lt = 2.0 * ORC_PI * p->R / (double)nt;
        double ls = 1.0 / fabs(f);
        for (int m = 0; m < 6; m++) {
            double len = (m == M_SF || m == M_SB) ? ls : lt;
            double q = round(one * len * (double)p->dir_mult[m] / 256.0);
            if (q < 1.0 || q * 255.0 / 16.0 >= (double)(1u << 26)) e = 3;
            c->len_q[m * nt + t] = (uint32_t)q;
        }
        c->cosq[t] = (int32_t)round(16384.0 * co);
        c->sinq[t] = (int32_t)round(16384.0 * s);
    }
    for (int m = 0; m < 6; m++) if (p->ct[m] >= (1u << 26)) e = 3;
    if (e) { orc_destroy(c); if (err) *err = e; return NULL; }
    if (err) *err = 0;
    return c;
}

void orc_set_threads(orc_ctx *c, int t)
{
#ifdef _OPENMP
    c->threads = t > 0 ? t : omp_get_max_threads();
#else
    (void)t; c->threads = 1;
#endif
}
int orc_get_threads(const orc_ctx *c) { return c->threads; }

const int32_t *orc_beta(const orc_ctx *c) { return c->beta; }
const uint8_t *orc_psi2(const orc_ctx *c) { return c->psi2; }
const uint8_t *orc_I(const orc_ctx *c) { return c->I; }
const int8_t *orc_J(const orc_ctx *c) { return c->J; }
const double *orc_K(const orc_ctx *c) { return c->K; }
const int32_t *orc_B(const orc_ctx *c) { return c->B; }
const uint32_t *orc_len_q(const orc_ctx *c) { return c->len_q; }
const int32_t *orc_cosq(const orc_ctx *c) { return c->cosq; }
const int32_t *orc_sinq(const orc_ctx *c) { return c->sinq; }

static inline int beta_k(const orc_ctx *c, int k, int t) { return c->beta[(t + k * (c->nt / 4)) & c->mt]; }

/* Curve maps.  Turn (m in LF,LB,RF,RB): thread (c0,c1) = (x',y'), sweep coordinate k = Theta,
 * eq (18) PAPER.md:266.  Straight: thread (c0,c1) = (x',Theta), sweep coordinate k = y',
 * eq (23) PAPER.md:291. */
void orc_curve_cell(const orc_ctx *c, int m, int c0, int c1, int k, int *i, int *j, int *th)
{
    if (m == M_LF || m == M_LB) {
        *i = (c0 + beta_k(c, 0, k)) & c->mx; *j = (c1 + beta_k(c, 3, k)) & c->mx; *th = k;
    } else if (m == M_RF || m == M_RB) {
        *i = (c0 + beta_k(c, 2, k)) & c->mx; *j = (c1 + beta_k(c, 1, k)) & c->mx; *th = k;
    } else {
        int b = c->B[(size_t)c1 * c->n + k];
        if (c->I[c1] == 0) { *i = k; *j = (c0 + b) & c->mx; }
        else { *i = (c0 + b) & c->mx; *j = k; }
        *th = c1;
    }
}

/* Maneuver edge maps, eq (25)-(31) PAPER.md:306-334 (eq (27) repaired per DESIGN R6). */
void orc_edge(const orc_ctx *c, int m, int i, int j, int t, int *i2, int *j2, int *t2)
{
    int mx = c->mx, mt = c->mt, n = c->n;
    int tp = (t + 1) & mt, tm = (t - 1) & mt;
    switch (m) {
    case M_LF: *i2 = (i + beta_k(c, 0, tp) - beta_k(c, 0, t)) & mx; *j2 = (j + beta_k(c, 3, tp) - beta_k(c, 3, t)) & mx; *t2 = tp; return;
    case M_LB: *i2 = (i + beta_k(c, 0, tm) - beta_k(c, 0, t)) & mx; *j2 = (j + beta_k(c, 3, tm) - beta_k(c, 3, t)) & mx; *t2 = tm; return;
    case M_RF: *i2 = (i + beta_k(c, 2, tm) - beta_k(c, 2, t)) & mx; *j2 = (j + beta_k(c, 1, tm) - beta_k(c, 1, t)) & mx; *t2 = tm; return;
    case M_RB: *i2 = (i + beta_k(c, 2, tp) - beta_k(c, 2, t)) & mx; *j2 = (j + beta_k(c, 1, tp) - beta_k(c, 1, t)) & mx; *t2 = tp; return;
    default: break;
    }
    /* straight: (30) is the + step of y', forward iff J >= 0 */
    int plus = ((m == M_SF) == (c->J[t] > 0));
    const int32_t *B = c->B + (size_t)t * n;
    *t2 = t;
    if (c->I[t] == 0) {
        int in = plus ? ((i + 1) & mx) : ((i - 1) & mx);
        *i2 = in; *j2 = (j + B[in] - B[i]) & mx;
    } else {
        int jn = plus ? ((j + 1) & mx) : ((j - 1) & mx);
        *j2 = jn; *i2 = (i + B[jn] - B[j]) & mx;
    }
}

static const int INV_M[6] = { M_LB, M_SB, M_RF, M_RB, M_SF, M_LF };

/* ------------------------------------------------------------------------------------------
 * Obstacle rendering ("rendering", l.226 wall, l.259 Psi offset, l.338).
 * Rasterisation rule = DESIGN R15 (ours; parity unpinned against the paper).
 * ---------------------------------------------------------------------------------------- */
static int covered(const orc_ctx *c, const orc_footprint *fp, int t, int da, int db)
{
    int64_t dx2 = 2 * (int64_t)da - c->psi2[t];                         /* eq (16): x = i + Psi0 */
    int64_t dy2 = 2 * (int64_t)db - c->psi2[(t + c->nt / 4) & c->mt];   /*          y = j + Psi1 */
    int64_t uq = dx2 * c->cosq[t] + dy2 * c->sinq[t];                    /* inverse of PAPER.md:86 */
    int64_t vq = -dx2 * c->sinq[t] + dy2 * c->cosq[t];
    int64_t ouq = (int64_t)round(fp->ou * 32768.0), ovq = (int64_t)round(fp->ov * 32768.0);
    int64_t p = floordiv(uq + ouq + 16384, 32768);
    int64_t q = floordiv(vq + ovq + 16384, 32768);
    if (p < 0 || p >= fp->mw || q < 0 || q >= fp->mh) return 0;
    return fp->mask[q * fp->mw + p] != 0;
}

int orc_footprint_radius(const orc_footprint *fp)
{
    double mu = fmax(fabs(-fp->ou - 0.5), fabs((double)fp->mw - 1.0 - fp->ou + 0.5));
    double mv = fmax(fabs(-fp->ov - 0.5), fabs((double)fp->mh - 1.0 - fp->ov + 0.5));
    return (int)ceil(hypot(mu, mv)) + 2;
}

/* One pose, brute force over every pixel of the bounding square. soft may be NULL. */
int orc_render_pose(const orc_ctx *c, const orc_footprint *fp, const uint8_t *hard, const uint8_t *soft,
                    int i, int j, int t, uint8_t *c_out, uint8_t *s_out)
{
    int rad = orc_footprint_radius(fp), n = c->n, mx = c->mx;
    if (2 * rad >= n) return -1;
    int blocked = (i == 0 || j == 0), s = 0;
    for (int db = -rad; db <= rad; db++)
        for (int da = -rad; da <= rad; da++) {
            if (!covered(c, fp, t, da, db)) continue;
            int a = (i + da) & mx, b = (j + db) & mx;
            if (a == 0 || b == 0 || hard[(size_t)b * n + a]) blocked = 1;
            if (soft && soft[(size_t)b * n + a] > s) s = soft[(size_t)b * n + a];
        }
    if (s < 16) s = 16;
    if (s > 255) s = 255;
    *c_out = (uint8_t)blocked;
    if (s_out) *s_out = (uint8_t)s;
    return 0;
}

/* Whole volume by brute force: C_out[idx] in {0,1}, S_out[idx] Q4.4 (may be NULL with soft). */
int orc_render_brute(const orc_ctx *c, const orc_footprint *fp, const uint8_t *hard, const uint8_t *soft,
                     uint8_t *C_out, uint8_t *S_out)
{
    int n = c->n, nt = c->nt;
    if (2 * orc_footprint_radius(fp) >= n) return -1;
#pragma omp parallel for num_threads(c->threads) schedule(static)
    for (int t = 0; t < nt; t++)
        for (int j = 0; j < n; j++)
            for (int i = 0; i < n; i++) {
                size_t idx = ((size_t)t * n + j) * n + i;
                uint8_t cc, ss;
                orc_render_pose(c, fp, hard, soft, i, j, t, &cc, &ss);
                C_out[idx] = cc;
                if (S_out) S_out[idx] = soft ? ss : 16;
            }
    return 0;
}

/* One Theta plane of orc_render_brute: the same per-pose definition (orc_render_pose) over all (i, j) of plane t and nothing
 * else, for whole-plane checks at sizes where the full brute-force volume takes too long.  C_out / S_out: n x n. */
int orc_render_brute_plane(const orc_ctx *c, const orc_footprint *fp, const uint8_t *hard, const uint8_t *soft, int t,
                           uint8_t *C_out, uint8_t *S_out)
{
    int n = c->n;
    if (2 * orc_footprint_radius(fp) >= n || t < 0 || t >= c->nt) return -1;
#pragma omp parallel for num_threads(c->threads) schedule(static)
    for (int j = 0; j < n; j++)
        for (int i = 0; i < n; i++) {
            uint8_t cc, ss;
            orc_render_pose(c, fp, hard, soft, i, j, t, &cc, &ss);
            C_out[(size_t)j * n + i] = cc;
            if (S_out) S_out[(size_t)j * n + i] = soft ? ss : 16;
        }
    return 0;
}

/* Area / orientation penalty on the obstacle volume ("direction and area-based velocity penalties"; "the
 * rendering ... handles any additional area and orientation related penalties", section VI l.338; Figure 19 l.463: "penalties
 * to inform the planner not to use the reverse direction lane").  The paper gives no formula: reading DESIGN R28.
 *   lane_dir[b][a]  preferred heading of pixel (a, b) in 1/256 turns (0 = +x, 64 = +y)
 *   lane_pen[b][a]  Q4.4 factor (16 = 1.0; values below 16 count as 16) on the reciprocal velocity of a vehicle that faces the
 *                   opposite way; in between the factor grows linearly with the angle
 * For the pose (i, j, Theta), evaluated at its own pixel (the rear-axle cell):
 *   h     = floor(256 Theta / N_theta)                      heading in 1/256 turns
 *   delta = min((h - dir) mod 256, (dir - h) mod 256)       0 .. 128
 *   f     = 16 + (((pen - 16) * 2 delta + 128) >> 8)        Q4.4, 16 .. pen
 *   S    <- min(255, (S * f + 8) >> 4)                      Q4.4 product, rounded half up
 * S: the rendered soft volume (R16), updated in place. */
void orc_apply_lane(const orc_ctx *c, uint8_t *S, const uint8_t *lane_dir, const uint8_t *lane_pen)
{
    int n = c->n, nt = c->nt;
    for (int t = 0; t < nt; t++) {
        int h = (int)(((int64_t)256 * t) / nt);
        for (int j = 0; j < n; j++)
            for (int i = 0; i < n; i++) {
                size_t px = (size_t)j * n + i, idx = ((size_t)t * n + j) * n + i;
                int pen = lane_pen[px] < 16 ? 16 : lane_pen[px];
                int d = (h - (int)lane_dir[px]) & 255;
                int delta = d < 256 - d ? d : 256 - d;
                int f = 16 + (((pen - 16) * 2 * delta + 128) >> 8);
                int s = ((int)S[idx] * f + 8) >> 4;
                S[idx] = (uint8_t)(s > 255 ? 255 : s);
            }
    }
}

/* Number of covered offsets for Theta (area check) and optional list output. */
int orc_footprint_offsets(const orc_ctx *c, const orc_footprint *fp, int t, int32_t *da_out, int32_t *db_out, int cap)
{
    int rad = orc_footprint_radius(fp), cnt = 0;
    for (int db = -rad; db <= rad; db++)
        for (int da = -rad; da <= rad; da++)
            if (covered(c, fp, t, da, db)) {
                if (da_out && cnt < cap) { da_out[cnt] = da; db_out[cnt] = db; }
                cnt++;
            }
    return cnt;
}

/* Same result as orc_render_brute, organised for full-size volumes: the covered offset set
 * depends only on (a-i, b-j, Theta) (it is a structuring element E_Theta); each row of E_Theta is
 * split into runs, the hard test of a run is a prefix-count difference and the soft max of a run is
 * a range-max query on a per-row sparse table.  Pinned against orc_render_brute in the tests. */
int orc_render_runs(const orc_ctx *c, const orc_footprint *fp, const uint8_t *hard, const uint8_t *soft,
                    uint8_t *C_out, uint8_t *S_out)
{
    int n = c->n, nt = c->nt, mx = c->mx;
    int rad = orc_footprint_radius(fp);
    if (2 * rad >= n) return -1;
    /* prefix counts of H = hard | wall over three periods of each row */
    int W = 3 * n;
    int32_t *PS = (int32_t *)malloc(sizeof(int32_t) * (size_t)n * (W + 1));
    for (int b = 0; b < n; b++) {
        int32_t *ps = PS + (size_t)b * (W + 1);
        ps[0] = 0;
        for (int x = 0; x < W; x++) {
            int a = x & mx;
            int h = (a == 0 || b == 0 || hard[(size_t)b * n + a]) ? 1 : 0;
            ps[x + 1] = ps[x] + h;
        }
    }
    /* sparse table of row maxima: ST[l][b][x] = max soft[b][(x .. x+2^l-1) & mx], x over 3 periods */
    int levels = 0;
    uint8_t *ST = NULL;
    if (soft && S_out) {
        while ((1 << (levels + 1)) <= 2 * rad + 1) levels++;
        levels += 1;
        ST = (uint8_t *)malloc((size_t)levels * n * W);
        for (int b = 0; b < n; b++)
            for (int x = 0; x < W; x++) ST[((size_t)0 * n + b) * W + x] = soft[(size_t)b * n + (x & mx)];
        for (int l = 1; l < levels; l++)
            for (int b = 0; b < n; b++) {
                const uint8_t *lo = ST + ((size_t)(l - 1) * n + b) * W;
                uint8_t *hi = ST + ((size_t)l * n + b) * W;
                int h = 1 << (l - 1);
                for (int x = 0; x < W; x++) {
                    uint8_t v = lo[x];
                    if (x + h < W && lo[x + h] > v) v = lo[x + h];
                    hi[x] = v;
                }
            }
    }
#pragma omp parallel for num_threads(c->threads) schedule(dynamic, 1)
    for (int t = 0; t < nt; t++) {
        /* runs of E_Theta: for each db the maximal intervals [a0,a1] of covered da */
        int side = 2 * rad + 1;
        int32_t *r_db = (int32_t *)malloc(sizeof(int32_t) * side * side);
        int32_t *r_a0 = (int32_t *)malloc(sizeof(int32_t) * side * side);
        int32_t *r_a1 = (int32_t *)malloc(sizeof(int32_t) * side * side);
        int nr = 0;
        for (int db = -rad; db <= rad; db++) {
            int da = -rad;
            while (da <= rad) {
                if (!covered(c, fp, t, da, db)) { da++; continue; }
                int a0 = da;
                while (da + 1 <= rad && covered(c, fp, t, da + 1, db)) da++;
                r_db[nr] = db; r_a0[nr] = a0; r_a1[nr] = da; nr++;
                da++;
            }
        }
        for (int j = 0; j < n; j++)
            for (int i = 0; i < n; i++) {
                size_t idx = ((size_t)t * n + j) * n + i;
                int blocked = (i == 0 || j == 0), s = 0;
                for (int r = 0; r < nr; r++) {
                    int b = (j + r_db[r]) & mx;
                    int x0 = n + i + r_a0[r], x1 = n + i + r_a1[r];
                    const int32_t *ps = PS + (size_t)b * (W + 1);
                    if (ps[x1 + 1] - ps[x0] > 0) blocked = 1;
                    if (ST) {
                        int len = x1 - x0 + 1, l = 0;
                        while ((2 << l) <= len) l++;
                        const uint8_t *st = ST + ((size_t)l * n + b) * W;
                        int v0 = st[x0], v1 = st[x1 - (1 << l) + 1];
                        if (v0 > s) s = v0;
                        if (v1 > s) s = v1;
                    }
                }
                if (s < 16) s = 16;
                C_out[idx] = (uint8_t)blocked;
                if (S_out) S_out[idx] = soft ? (uint8_t)s : 16;
            }
        free(r_db); free(r_a0); free(r_a1);
    }
    free(PS); free(ST);
    return 0;
}

/* ------------------------------------------------------------------------------------------
 * Kernel-style processing (section VIII.B; the loop body is Insert 5,
 * PAPER.md:946-949, "identical to the basic loop"; v starts at infinity as in Insert 3 l.923,
 * DESIGN R2; blocked vertices are removed, DESIGN R10; the obstacle value of
 * the SOURCE vertex multiplies the edge length, PAPER.md:338 + l.949, DESIGN R7).
 * ---------------------------------------------------------------------------------------- */
static inline uint32_t edge_w(const orc_ctx *c, const uint8_t *S, int m, int t, size_t idx)
{
    uint32_t s = S ? S[idx] : 16u;
    return (uint32_t)(((uint64_t)c->len_q[m * c->nt + t] * s) >> 4);
}

static void sweep_curve(const orc_ctx *c, int m, uint32_t *V, const uint8_t *C, const uint8_t *S, int c0, int c1)
{
    int n = c->n, nt = c->nt;
    uint32_t ct = c->p.ct[m], v = ORC_INF;
    int turn = !(m == M_SF || m == M_SB);
    int steps, up;
    if (turn) { steps = 2 * nt; up = (m == M_LF || m == M_RB); }           /* two full loops, l.356 */
    else { steps = n; up = ((m == M_SF) == (c->J[c1] > 0)); }             /* one, direction l.294 */
    int len = turn ? nt : n;
    for (int s = 0; s < steps; s++) {
        int k = up ? (s % len) : (len - 1 - (s % len));
        int i, j, t;
        orc_curve_cell(c, m, c0, c1, k, &i, &j, &t);
        size_t idx = ((size_t)t * n + j) * n + i;
        if (C[idx]) { v = ORC_INF; continue; }
        uint32_t u = V[idx];
        V[idx] = v < u ? v : u;                          /* V[i] = min(v,u)            l.948 */
        uint32_t uc = cadd(u, ct);
        v = cadd(v < uc ? v : uc, edge_w(c, S, m, t, idx)); /* v = min(v,u+ct)+cx*B[i] l.949 */
    }
}

/* One maneuver kernel = all curves of maneuver m. Curves are disjoint (l.224). */
void orc_sweep(const orc_ctx *c, int m, uint32_t *V, const uint8_t *C, const uint8_t *S)
{
    int n = c->n, nt = c->nt;
    int turn = !(m == M_SF || m == M_SB);
    int n1 = turn ? n : nt;
#pragma omp parallel for num_threads(c->threads) schedule(static)
    for (int c1 = 0; c1 < n1; c1++)
        for (int c0 = 0; c0 < n; c0++) sweep_curve(c, m, V, C, S, c0, c1);
}

/* Cycle order LF, SF, RB, RF, SB, LB; FORWARD_ONLY keeps LF, SF, RF (Dubins car, l.681). */
void orc_cycles(const orc_ctx *c, uint32_t *V, const uint8_t *C, const uint8_t *S, int ncycles)
{
    for (int k = 0; k < ncycles; k++)
        for (int m = 0; m < 6; m++) {
            if ((c->p.flags & ORC_FLAG_FORWARD_ONLY) && (m == M_RB || m == M_SB || m == M_LB)) continue;
            orc_sweep(c, m, V, C, S);
        }
}

/* V <- INF, V[start] <- 0, then ncycles maneuver cycles. Returns -4 if the start is blocked. */
int orc_run(const orc_ctx *c, uint32_t *V, const uint8_t *C, const uint8_t *S, int si, int sj, int st, int ncycles)
{
    size_t nr = (size_t)c->n * c->n * c->nt;
    size_t sidx = ((size_t)st * c->n + sj) * c->n + si;
    if (si < 0 || sj < 0 || st < 0 || si >= c->n || sj >= c->n || st >= c->nt) return -1;
    if (C[sidx]) return -4;
    for (size_t x = 0; x < nr; x++) V[x] = ORC_INF;
    V[sidx] = 0;
    orc_cycles(c, V, C, S, ncycles);
    return 0;
}

/* ------------------------------------------------------------------------------------------
 * Dijkstra on the graph defined by the edge maps (25)-(31) plus S(X).
 * kind 0: Star S(X), 7 vertices / 18 edges per X (Table 1 l.437);
 * kind 1: Compact, 3 vertices / 10 edges per X (Table 1 l.436), needs conforming
 *         weights: ct[SF]=ct[SB]=0, ct[LF]=ct[LB], ct[RF]=ct[RB].
 * Vout[X] = value of the transition vertex (Star) / straight vertex (Compact).
 * ---------------------------------------------------------------------------------------- */
typedef struct { uint32_t d; uint64_t v; } hitem;
typedef struct { hitem *a; size_t n, cap; } heap;
static void hpush(heap *h, uint32_t d, uint64_t v)
{
    if (h->n == h->cap) { h->cap = h->cap ? 2 * h->cap : 1024; h->a = (hitem *)realloc(h->a, h->cap * sizeof(hitem)); }
    size_t k = h->n++;
    while (k > 0) {
        size_t p = (k - 1) / 2;
        if (h->a[p].d <= d) break;
        h->a[k] = h->a[p]; k = p;
    }
    h->a[k].d = d; h->a[k].v = v;
}
static hitem hpop(heap *h)
{
    hitem top = h->a[0], last = h->a[--h->n];
    size_t k = 0;
    for (;;) {
        size_t l = 2 * k + 1, r = l + 1, s;
        if (l >= h->n) break;
        s = (r < h->n && h->a[r].d < h->a[l].d) ? r : l;
        if (h->a[s].d >= last.d) break;
        h->a[k] = h->a[s]; k = s;
    }
    if (h->n) h->a[k] = last;
    return top;
}

/* Instrumentation for the structural pin of Table 1 (k_V vertices and k_E edges per X):
 * while a probe cell is set, the next Dijkstra run counts the vertices of that cell it settles and the edges it relaxes
 * out of them.  Counting only: the search itself is untouched. */
static size_t g_probe_X = (size_t)-1;
static int g_probe_vertices = 0, g_probe_edges = 0;
void orc_dijkstra_probe(const orc_ctx *c, int i, int j, int t)
{
    g_probe_X = (i < 0) ? (size_t)-1 : ((size_t)t * c->n + j) * c->n + i;
    g_probe_vertices = g_probe_edges = 0;
}
void orc_dijkstra_probe_result(int *vertices, int *edges) { *vertices = g_probe_vertices; *edges = g_probe_edges; }

int orc_dijkstra_from(const orc_ctx *c, int kind, const uint8_t *C, const uint8_t *S, int si, int sj, int st, int m0, uint32_t *Vout)
{
    int n = c->n, nt = c->nt;
    size_t nr = (size_t)n * n * nt;
    int fwd_only = c->p.flags & ORC_FLAG_FORWARD_ONLY;
    const uint32_t *ct = c->p.ct;
    if (kind == 1 && !(ct[M_SF] == 0 && ct[M_SB] == 0 && ct[M_LF] == ct[M_LB] && ct[M_RF] == ct[M_RB])) return -1;
    int nv = kind == 0 ? 7 : 3;
    size_t sidx = ((size_t)st * n + sj) * n + si;
    if (C[sidx]) return -4;
    uint32_t *D = (uint32_t *)malloc(sizeof(uint32_t) * nr * nv);
    for (size_t x = 0; x < nr * nv; x++) D[x] = ORC_INF;
    heap h = { 0, 0, 0 };
    D[sidx * nv] = 0;
    hpush(&h, 0, (uint64_t)sidx * nv);
    if (m0 >= 0) {                                          /* maneuver m0 is in progress at the start: */
        if (kind != 0 || m0 > 5) { free(D); return -1; }    /* its Star vertex is a source too, so continuing it costs no c_t */
        D[sidx * nv + 1 + m0] = 0;
        hpush(&h, 0, (uint64_t)sidx * nv + 1 + m0);
    }
#define RELAX(vid, nd) do { uint32_t nd_ = (nd); uint64_t v_ = (vid); g_probe_edges += probing; if (nd_ < D[v_]) { D[v_] = nd_; hpush(&h, nd_, v_); } } while (0)
    while (h.n) {
        hitem it = hpop(&h);
        if (it.d != D[it.v]) continue;
        size_t X = it.v / nv; int k = (int)(it.v % nv);
        const int probing = (X == g_probe_X);
        g_probe_vertices += probing;
        int i = (int)(X % n), j = (int)((X / n) % n), t = (int)(X / ((size_t)n * n));
        if (kind == 0) {
            if (k == 0) {                                   /* transition vertex: T -> (X,m), cost ct[m] */
                for (int m = 0; m < 6; m++) {
                    if (fwd_only && (m == M_RB || m == M_SB || m == M_LB)) continue;
                    RELAX(X * 7 + 1 + m, cadd(it.d, ct[m]));
                }
            } else {
                int m = k - 1, i2, j2, t2;
                RELAX(X * 7, it.d);                          /* (X,m) -> T, free (DESIGN R8) */
                orc_edge(c, m, i, j, t, &i2, &j2, &t2);
                size_t X2 = ((size_t)t2 * n + j2) * n + i2;
                if (!C[X2]) RELAX(X2 * 7 + k, cadd(it.d, edge_w(c, S, m, t, X)));
            }
        } else {
            /* k: 0 = STRAIGHT (= transition state), 1 = LEFT, 2 = RIGHT */
            static const int MF[3] = { M_SF, M_LF, M_RF }, MB[3] = { M_SB, M_LB, M_RB };
            if (k == 0) { RELAX(X * 3 + 1, cadd(it.d, ct[M_LF])); RELAX(X * 3 + 2, cadd(it.d, ct[M_RF])); }
            else RELAX(X * 3, it.d);
            for (int d = 0; d < 2; d++) {
                int m = d == 0 ? MF[k] : MB[k], i2, j2, t2;
                if (d == 1 && fwd_only) continue;
                orc_edge(c, m, i, j, t, &i2, &j2, &t2);
                size_t X2 = ((size_t)t2 * n + j2) * n + i2;
                if (!C[X2]) RELAX(X2 * 3 + k, cadd(it.d, edge_w(c, S, m, t, X)));
            }
        }
    }
#undef RELAX
    for (size_t x = 0; x < nr; x++) Vout[x] = D[x * nv];
    free(D); free(h.a);
    return 0;
}

/* ------------------------------------------------------------------------------------------
 * Back-tracking (eq (32)): repeated reverse Bellman step over the six whole
 * curves through the current vertex.  Tie rule DESIGN R19: candidates are visited in cycle
 * order, then by increasing distance, and only a strictly smaller value replaces the best.
 * out[0] = goal ... out[count-1] = start; *cost = sum over the plan's segments of ct[m] + edge weights
 * (= V[goal] once the volume has converged, <= V[goal] before).  Returns 0, -5 goal unreached,
 * -6 buffer too small.
 * ---------------------------------------------------------------------------------------- */
/* m0 >= 0: maneuver m0 was in progress at the start (orc_run_from): the segment that leaves the START under m0
 * carries no transition cost */
int orc_backtrack_from(const orc_ctx *c, const uint32_t *V, const uint8_t *C, const uint8_t *S,
                       int si, int sj, int st, int m0, int gi, int gj, int gt,
                       orc_waypoint *out, int cap, int *count, uint32_t *cost)
{
    int n = c->n, nt = c->nt, cnt = 0;
    int fwd_only = c->p.flags & ORC_FLAG_FORWARD_ONLY;
    int ci = gi, cj = gj, cth = gt;
    uint32_t total = 0;                    /* plan cost = sum over segments of ct[m] + E_sum (eq (32)) */
    *count = 0; *cost = ORC_INF;
    size_t gidx = ((size_t)gt * n + gj) * n + gi;
    if (C[gidx]) return -5;
    if (gi == si && gj == sj && gt == st) {
        if (cap < 1) return -6;
        out[0].i = gi; out[0].j = gj; out[0].theta = gt; out[0].m = -1;
        *count = 1; *cost = 0; return 0;
    }
    for (;;) {
        uint32_t best = ORC_INF, bseg = 0; int bi = 0, bj = 0, bt = 0, bm = -1;
        for (int m = 0; m < 6; m++) {
            if (fwd_only && (m == M_RB || m == M_SB || m == M_LB)) continue;
            int turn = !(m == M_SF || m == M_SB);
            int maxk = turn ? nt - 1 : n;
            int pi = ci, pj = cj, pt = cth;
            uint32_t E = 0;
            for (int k = 1; k <= maxk; k++) {
                int qi, qj, qt;
                orc_edge(c, INV_M[m], pi, pj, pt, &qi, &qj, &qt);   /* one step against m (l.306: inverse map) */
                size_t q = ((size_t)qt * n + qj) * n + qi;
                if (C[q]) break;
                E = cadd(E, edge_w(c, S, m, qt, q));
                uint32_t ctm = (m == m0 && qi == si && qj == sj && qt == st) ? 0 : c->p.ct[m];
                uint32_t cand = cadd(cadd(V[q], ctm), E);
                if (cand < best) { best = cand; bseg = cadd(ctm, E); bi = qi; bj = qj; bt = qt; bm = m; }
                pi = qi; pj = qj; pt = qt;
            }
        }
        if (best == ORC_INF) return -5;
        total = cadd(total, bseg);
        if (cnt >= cap) return -6;
        out[cnt].i = ci; out[cnt].j = cj; out[cnt].theta = cth; out[cnt].m = bm; cnt++;
        ci = bi; cj = bj; cth = bt;
        if (ci == si && cj == sj && cth == st) break;
    }
    if (cnt >= cap) return -6;
    out[cnt].i = ci; out[cnt].j = cj; out[cnt].theta = cth; out[cnt].m = -1; cnt++;
    *count = cnt; *cost = total;
    return 0;
}

int orc_backtrack(const orc_ctx *c, const uint32_t *V, const uint8_t *C, const uint8_t *S,
                  int si, int sj, int st, int gi, int gj, int gt,
                  orc_waypoint *out, int cap, int *count, uint32_t *cost)
{
    return orc_backtrack_from(c, V, C, S, si, sj, st, -1, gi, gj, gt, out, cap, count, cost);
}

int orc_dijkstra(const orc_ctx *c, int kind, const uint8_t *C, const uint8_t *S, int si, int sj, int st, uint32_t *Vout)
{
    return orc_dijkstra_from(c, kind, C, S, si, sj, st, -1, Vout);
}

/* Start state with a maneuver in progress (section XII: "if a maneuver is in progress, there should be
 * no transition cost to start with that maneuver, which is easily accomplished by using the appropriate start
 * configuration").  Reading DESIGN R26: besides V[start] = 0 the vertices AHEAD of the start on the curve of m0 are
 * seeded with the summed edge weights from the start (no c_t), up to the first blocked vertex (at most one lap);
 * then the cycles run as usual.  The walk uses the edge maps (25)-(31), not the sweep code. */
int orc_run_from(const orc_ctx *c, uint32_t *V, const uint8_t *C, const uint8_t *S, int si, int sj, int st, int m0, int ncycles)
{
    int n = c->n, nt = c->nt;
    size_t nr = (size_t)n * n * nt;
    size_t sidx = ((size_t)st * n + sj) * n + si;
    if (si < 0 || sj < 0 || st < 0 || si >= n || sj >= n || st >= nt || m0 < -1 || m0 > 5) return -1;
    if (m0 >= 0 && (c->p.flags & ORC_FLAG_FORWARD_ONLY) && (m0 == M_RB || m0 == M_SB || m0 == M_LB)) return -1;
    if (C[sidx]) return -4;
    for (size_t x = 0; x < nr; x++) V[x] = ORC_INF;
    V[sidx] = 0;
    if (m0 >= 0) {
        int i = si, j = sj, t = st, steps = (m0 == M_SF || m0 == M_SB) ? n : nt - 1;
        uint32_t acc = 0;
        for (int k = 0; k < steps; k++) {
            int i2, j2, t2;
            size_t X = ((size_t)t * n + j) * n + i;
            orc_edge(c, m0, i, j, t, &i2, &j2, &t2);
            size_t X2 = ((size_t)t2 * n + j2) * n + i2;
            if (C[X2]) break;
            acc = cadd(acc, edge_w(c, S, m0, t, X));
            if (acc < V[X2]) V[X2] = acc;
            i = i2; j = j2; t = t2;
        }
    }
    orc_cycles(c, V, C, S, ncycles);
    return 0;
}

/* ------------------------------------------------------------------------------------------------
 * Steps 1-2 of the pipeline (section VII l.342): "distance transform obstacle image
 * and calculate new obstacle image as a function of distance".  The paper leaves the function open
 * ("some function of the distance"); reading DESIGN R17:
 *     H     = hard | wall (row 0 and column 0), NOT toroidal (as the scene generators do)
 *     d2    = exact squared Euclidean distance of a pixel centre to the nearest pixel centre of H
 *     d     = sqrtf(d2)                                   float32, correctly rounded
 *     soft  = clamp(rintf(16 * (1 + k / (d + 1))), 16, 255)  float32 operation by operation (no FMA), Q4.4
 * Plain definition written out: for every pixel the minimum over ALL hard pixels (orc_edt_brute, O(N^4),
 * tiny images only), and the exact separable form min over x' of (x - x')^2 + g(y, x')^2 with g = distance
 * to the nearest hard pixel in column x' (orc_soft_from_hard, O(N^3)).  Pins: the two agree; both agree
 * with scipy.ndimage.distance_transform_edt (tests/test_oracle_dt.py).
 * ------------------------------------------------------------------------------------------------ */
#define ORC_DT_FAR 20000            /* "no hard pixel in this column": FAR^2 + N^2 < 2^31 for N <= 4096 */

static int dt_hard(const uint8_t *hard, int n, int x, int y) { return hard[(size_t)y * n + x] != 0 || x == 0 || y == 0; }

void orc_edt_brute(const uint8_t *hard, int n, int32_t *d2_out)
{
    for (int y = 0; y < n; y++)
        for (int x = 0; x < n; x++) {
            int64_t best = INT64_MAX;
            for (int b = 0; b < n; b++)
                for (int a = 0; a < n; a++)
                    if (dt_hard(hard, n, a, b)) {
                        int64_t d = (int64_t)(x - a) * (x - a) + (int64_t)(y - b) * (y - b);
                        if (d < best) best = d;
                    }
            d2_out[(size_t)y * n + x] = (int32_t)best;
        }
}

/* d2_out (int32, may be NULL), dist_out (float, may be NULL), soft_out (uint8, may be NULL): n x n each */
int orc_soft_from_hard(const uint8_t *hard, int n, float k, int32_t *d2_out, float *dist_out, uint8_t *soft_out)
{
    int32_t *g = (int32_t *)malloc(sizeof(int32_t) * (size_t)n * n);
    if (!g) return -1;
    for (int x = 0; x < n; x++) {                      /* nearest hard pixel in the same column */
        for (int y = 0; y < n; y++) {
            int best = ORC_DT_FAR;
            for (int b = 0; b < n; b++)
                if (dt_hard(hard, n, x, b)) { int d = y > b ? y - b : b - y; if (d < best) best = d; }
            g[(size_t)y * n + x] = best;
        }
    }
#pragma omp parallel for schedule(static)
    for (int y = 0; y < n; y++)
        for (int x = 0; x < n; x++) {
            int64_t best = INT64_MAX;
            for (int a = 0; a < n; a++) {
                int64_t gg = g[(size_t)y * n + a];
                int64_t d = (int64_t)(x - a) * (x - a) + gg * gg;
                if (d < best) best = d;
            }
            const size_t idx = (size_t)y * n + x;
            if (d2_out) d2_out[idx] = (int32_t)best;
            volatile float d = sqrtf((float)best);     /* volatile: one rounding per operation, no contraction */
            volatile float den = d + 1.0f;
            volatile float q = k / den;
            volatile float s = 1.0f + q;
            volatile float v = 16.0f * s;
            float r = rintf(v);
            if (dist_out) dist_out[idx] = d;
            if (soft_out) soft_out[idx] = (uint8_t)(r < 16.0f ? 16.0f : r > 255.0f ? 255.0f : r);
        }
    free(g);
    return 0;
}

/* ------------------------------------------------------------------------------------------------
 * Goal search, step 6 of the pipeline (section IX l.372-374): "more than one configuration
 * in the goal set and ... a reward function (such as a function of difference to the ideal pose) over them.
 * The optimization criterion is the reward for the vertex minus the cost to get there ... Multiple ideal
 * goals is also possible".  Appendix G (l.1169) names the parameters: d "radius in number of grid cells",
 * W, w "weights for goal search".  Reading DESIGN R20 (the paper gives no formula):
 *   goal set of an ideal goal (gi, gj, gt) = vertices (gi+di, gj+dj, (gt+dt) mod N_theta) with di^2 + dj^2 <= d^2,
 *   |dt| <= d, inside the grid (no spatial wrap), not blocked and reached (V != INF);
 *   reward = -(W (di^2 + dj^2) + w dt^2) in cost units, so the criterion is  min  V + W (di^2 + dj^2) + w dt^2;
 *   ties: first in the order (goal index, dt, dj, di), each ascending.
 * Returns 0 and fills out[0..2] = (i, j, theta), out[3] = index of the ideal goal, *score; -5 if the set is empty.
 * ------------------------------------------------------------------------------------------------ */
int orc_goal_search(const orc_ctx *c, const uint32_t *V, const int32_t *goals, int n_goals, int d, uint32_t W, uint32_t w,
                    int32_t *out, uint64_t *score)
{
    const int n = c->n, nt = c->nt;
    uint64_t best = UINT64_MAX;
    for (int g = 0; g < n_goals; g++)
        for (int dt = -d; dt <= d; dt++)
            for (int dj = -d; dj <= d; dj++)
                for (int di = -d; di <= d; di++) {
                    if (di * di + dj * dj > d * d) continue;
                    const int i = goals[3 * g] + di, j = goals[3 * g + 1] + dj, t = (goals[3 * g + 2] + dt + 4 * nt) % nt;
                    if (i < 0 || i >= n || j < 0 || j >= n) continue;
                    const uint32_t v = V[((size_t)t * n + j) * n + i];
                    if (v == ORC_INF) continue;
                    const uint64_t s = (uint64_t)v + (uint64_t)W * (uint64_t)(di * di + dj * dj) + (uint64_t)w * (uint64_t)(dt * dt);
                    if (s < best) { best = s; out[0] = i; out[1] = j; out[2] = t; out[3] = g; }
                }
    if (best == UINT64_MAX) return -5;
    *score = best;
    return 0;
}

/* ------------------------------------------------------------------------------------------------
 * Reachability ("bit-vector") planner, appendix C: edge weights zero on maneuver edges
 * (infinite at obstacles), one on transition edges; "the value of a vertex during maneuver processing can be
 * represented by a single bit.  That bit indicates ... if the vertex can be reached in m maneuvers or less".
 * "The maneuver kernels now read from the previous reachability volume (at m maneuvers) ... and produce the
 * reachability of one of the volumes of maneuver vertices (at m maneuvers plus that maneuver), which is combined
 * ... into the reachability of the transition vertices (at m + 1 maneuvers)" -- a Jacobi step per level; the loop
 * body is Insert 2 (l.873-878): v &= Vi[i]; Vo[i] = v; v |= B[i]  (their bit is 0 = reachable; here 1 = reachable:
 * v |= Li[i]; blocked -> v = 0, else Lo[i] |= v).  Blocked vertices are removed (DESIGN R10).  "The output
 * reachability bit volumes are kept around to support back-tracking" (l.897).
 * The oracle keeps one byte per vertex: K[X] = smallest m with X reachable in <= m maneuvers, 255 = not within
 * n_levels (n_levels <= 254).  The level volumes are L_m = (K <= m).
 * ------------------------------------------------------------------------------------------------ */
static void reach_sweep(const orc_ctx *c, int m, const uint8_t *K, uint8_t *Knew, const uint8_t *C, int level)
{
    int n = c->n, nt = c->nt;
    int turn = !(m == M_SF || m == M_SB);
    int n1 = turn ? n : nt, len = turn ? nt : n;
#pragma omp parallel for num_threads(c->threads) schedule(static)
    for (int c1 = 0; c1 < n1; c1++)
        for (int c0 = 0; c0 < n; c0++) {
            int steps, up;
            if (turn) { steps = 2 * nt; up = (m == M_LF || m == M_RB); }          /* two full loops, l.356 */
            else { steps = n; up = ((m == M_SF) == (c->J[c1] > 0)); }
            int v = 0;
            for (int s = 0; s < steps; s++) {
                int k = up ? (s % len) : (len - 1 - (s % len)), i, j, t;
                orc_curve_cell(c, m, c0, c1, k, &i, &j, &t);
                size_t idx = ((size_t)t * n + j) * n + i;
                if (C[idx]) { v = 0; continue; }
                if (K[idx] <= level) v = 1;                      /* reachable at <= level maneuvers: v |= Li[i] */
                if (v && Knew[idx] > level + 1) Knew[idx] = (uint8_t)(level + 1);
            }
        }
}

int orc_reach_run(const orc_ctx *c, uint8_t *K, const uint8_t *C, int si, int sj, int st, int n_levels)
{
    int n = c->n, nt = c->nt;
    size_t nr = (size_t)n * n * nt, sidx = ((size_t)st * n + sj) * n + si;
    int fwd_only = c->p.flags & ORC_FLAG_FORWARD_ONLY;
    if (si < 0 || sj < 0 || st < 0 || si >= n || sj >= n || st >= nt || n_levels < 0 || n_levels > 254) return -1;
    if (C[sidx]) return -4;
    uint8_t *Kn = (uint8_t *)malloc(nr);
    if (!Kn) return -7;
    memset(K, 255, nr);
    K[sidx] = 0;
    for (int level = 0; level < n_levels; level++) {
        memcpy(Kn, K, nr);
        for (int m = 0; m < 6; m++) {
            if (fwd_only && (m == M_RB || m == M_SB || m == M_LB)) continue;
            reach_sweep(c, m, K, Kn, C, level);                  /* all six read level m, write level m + 1 */
        }
        memcpy(K, Kn, nr);
    }
    free(Kn);
    return 0;
}

/* Back-tracking over the level volumes: from the goal at its level k, the maneuvers in cycle order; for each, walk
 * back along its curve (against its direction) until a blocked vertex; the first vertex reachable at <= k - 1
 * maneuvers is that maneuver's candidate; the first maneuver with a candidate wins (DESIGN R27).  Records as in
 * orc_backtrack; *cost = number of maneuvers. */
int orc_reach_backtrack(const orc_ctx *c, const uint8_t *K, const uint8_t *C, int si, int sj, int st, int gi, int gj, int gt,
                        orc_waypoint *out, int cap, int *count, uint32_t *cost)
{
    int n = c->n, nt = c->nt, cnt = 0;
    int fwd_only = c->p.flags & ORC_FLAG_FORWARD_ONLY;
    int ci = gi, cj = gj, cth = gt;
    *count = 0; *cost = ORC_INF;
    size_t gidx = ((size_t)gt * n + gj) * n + gi;
    if (C[gidx] || K[gidx] == 255) return -5;
    const int total = K[gidx];
    while (!(ci == si && cj == sj && cth == st)) {
        int k = K[((size_t)cth * n + cj) * n + ci], found = 0, bi = 0, bj = 0, bt = 0, bm = -1;
        if (k == 0 || k == 255) return -5;
        for (int m = 0; m < 6 && !found; m++) {
            if (fwd_only && (m == M_RB || m == M_SB || m == M_LB)) continue;
            int maxk = (m == M_SF || m == M_SB) ? n : nt - 1;
            int pi = ci, pj = cj, pt = cth;
            for (int s = 1; s <= maxk; s++) {
                int qi, qj, qt;
                orc_edge(c, INV_M[m], pi, pj, pt, &qi, &qj, &qt);
                size_t q = ((size_t)qt * n + qj) * n + qi;
                if (C[q]) break;
                if (K[q] <= k - 1) { found = 1; bi = qi; bj = qj; bt = qt; bm = m; break; }
                pi = qi; pj = qj; pt = qt;
            }
        }
        if (!found) return -5;
        if (cnt >= cap) return -6;
        out[cnt].i = ci; out[cnt].j = cj; out[cnt].theta = cth; out[cnt].m = bm; cnt++;
        ci = bi; cj = bj; cth = bt;
    }
    if (cnt >= cap) return -6;
    out[cnt].i = ci; out[cnt].j = cj; out[cnt].theta = cth; out[cnt].m = -1; cnt++;
    *count = cnt; *cost = (uint32_t)total;
    return 0;
}
