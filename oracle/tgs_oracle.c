/*
 * tgs_oracle.c -- CPU ORACLE for the TurboGS sparse-pixel rasterisation hot path.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may build, load or call it.  It
 * shares no code, header, table or helper with the CUDA path
 * (paper_2606_15924_b200/csrc); the only thing both sides consume is the seeded input
 * generator in workloads/.
 *
 * Plain, slow, single-threaded C.  One source, two builds:
 *     -DORC_F64  : real = double  (finite-difference pins, cross-check of the fp32 build)
 *     (default)  : real = float   (the parity referee: the path's discrete decisions --
 *                  tile rects, depth keys, the alpha / transmittance thresholds -- are
 *                  taken in fp32, BASELINE.json north_star "fp32"; DESIGN.md "Readings" R0)
 * Compile with -O2 -ffp-contract=off: every +,-,*,/ below is rounded once, in the order
 * written (left to right); the only fused operations are the explicit rfma() calls.
 *
 * What it computes, step by step (citations: PAPER.md = /root/reference/PAPER.md, the
 * paper text; SURVEY.md section 8c lists the readings taken where the paper is silent):
 *   O1 orc_preprocess   EWA projection, conic, radius, tile rect, SH colour
 *   O2 orc_bin_sort     (tile, depth, id)-ordered pair list + CSR ranges      PAPER.md:64  K(p)
 *   O3 orc_sample       per-tile error, top-k tiles, tile-ordered pixel CSR   PAPER.md:73, 93 (Eq.2),
 *                                                                            128-150, 156
 *   O4 orc_raster_fwd   Eq. 1 alpha compositing on the sampled pixels         PAPER.md:66 (Eq.1), 154-166
 *   O5 orc_raster_bwd   exact derivative of O4
 *   O6 orc_project_bwd  chain through O1 to (mu, s, q, sh)
 *   O7 orc_loss_sparse  Charbonnier + tile-level sparse NCC + lambda_ncc      PAPER.md:168-208 (Eq.9-11),
 *                                                                            472-481 (Eq.17-18)
 * Pins (tests/test_oracle_pins.py): closed-form isotropic render, two-Gaussian
 * compositing, partition of unity, transmittance monotonicity, SH orthonormality by
 * quadrature, brute-force binning, full mask == dense, empty mask == zero gradients,
 * colour-linearity identity, fp64 central finite differences; O7: numpy corrcoef definition,
 * affine invariances of NCC, Charbonnier closed forms, both lambda regimes, finite differences.  No function here is
 * "parity unpinned".
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#ifdef ORC_F64
typedef double real;
#define rsqrt_ sqrt
#define rfloor floor
#define rceil ceil
#define rexp exp
#define rabs fabs
#define rfma fma
#else
typedef float real;
#define rsqrt_ sqrtf
#define rfloor floorf
#define rceil ceilf
#define rexp expf
#define rabs fabsf
#define rfma fmaf
#endif
#define K_(x) ((real)(x))

/* ---- named constants (SURVEY.md 8c readings 2, 3: the paper is silent, these are the
 *      constants of the "original rasterization kernels" it modifies) ---- */
#define TILE 16
#define LOWPASS K_(0.3)                 /* EWA low-pass dilation added to the 2D covariance */
#define JCLAMP K_(1.3)                  /* Jacobian clamp: |t_x/t_z| <= 1.3 tan(fov_x/2)     */
#define RADIUS_SIGMAS K_(3.0)
#define LAMBDA_GUARD K_(0.1)
#define ALPHA_MIN K_(0.00392156862745098) /* 1/255 */
#define ALPHA_MAX K_(0.99)
#define T_MIN K_(0.0001)
#define ERR_CLAMP K_(15.999)
#define ERR_SCALE K_(1048576.0)         /* 2^20 */

/* real SH basis constants */
#define SH_C0 K_(0.28209479177387814)
#define SH_C1 K_(0.4886025119029199)
#define SH_C2A K_(1.0925484305920792)
#define SH_C2B K_(0.31539156525252005)
#define SH_C2C K_(0.5462742152960396)
#define SH_C3A K_(0.5900435899266435)
#define SH_C3B K_(2.890611442640554)
#define SH_C3C K_(0.4570457994644658)
#define SH_C3D K_(0.3731763325901154)
#define SH_C3E K_(1.445305721320277)

typedef struct {
    int32_t W, H;
    real fx, fy, cx, cy;
    real Rcw[9]; /* world->camera rotation, row-major */
    real tau[3]; /* world->camera translation */
    real znear;
    real bg[3];
} orc_cam;

static real rmin(real a, real b) { return a < b ? a : b; }
static real rmax(real a, real b) { return a > b ? a : b; }
static int imin(int a, int b) { return a < b ? a : b; }

int orc_real_bytes(void) { return (int)sizeof(real); }

/* q = (w,x,y,z) -> rotation matrix, as the quadratic polynomial (no normalisation inside). */
static void quat_to_R(const real* q, real R[9]) {
    real w = q[0], x = q[1], y = q[2], z = q[3];
    R[0] = K_(1.0) - K_(2.0) * (y * y + z * z);
    R[1] = K_(2.0) * (x * y - w * z);
    R[2] = K_(2.0) * (x * z + w * y);
    R[3] = K_(2.0) * (x * y + w * z);
    R[4] = K_(1.0) - K_(2.0) * (x * x + z * z);
    R[5] = K_(2.0) * (y * z - w * x);
    R[6] = K_(2.0) * (x * z - w * y);
    R[7] = K_(2.0) * (y * z + w * x);
    R[8] = K_(1.0) - K_(2.0) * (x * x + y * y);
}
void orc_quat_to_R(const real* q, real* R) { quat_to_R(q, R); }

/* Sigma = M M^T, M = R diag(s).  Returns the full symmetric 3x3. */
static void cov3d(const real* s, const real* q, real Sg[9], real R[9]) {
    real M[9];
    quat_to_R(q, R);
    for (int r = 0; r < 3; ++r)
        for (int c = 0; c < 3; ++c) M[3 * r + c] = R[3 * r + c] * s[c];
    for (int r = 0; r < 3; ++r)
        for (int c = 0; c < 3; ++c)
            Sg[3 * r + c] = M[3 * r + 0] * M[3 * c + 0] + M[3 * r + 1] * M[3 * c + 1] + M[3 * r + 2] * M[3 * c + 2];
}
void orc_cov3d(const real* s, const real* q, real* Sg) { real R[9]; cov3d(s, q, Sg, R); }

/* The 16 real SH basis functions of degree <= 3 at unit direction d. */
static void sh_basis(const real* d, real B[16]) {
    real x = d[0], y = d[1], z = d[2];
    real xx = x * x, yy = y * y, zz = z * z, xy = x * y, yz = y * z, xz = x * z;
    B[0] = SH_C0;
    B[1] = (-SH_C1) * y;
    B[2] = SH_C1 * z;
    B[3] = (-SH_C1) * x;
    B[4] = SH_C2A * xy;
    B[5] = (-SH_C2A) * yz;
    B[6] = SH_C2B * ((K_(2.0) * zz - xx) - yy);
    B[7] = (-SH_C2A) * xz;
    B[8] = SH_C2C * (xx - yy);
    B[9] = ((-SH_C3A) * y) * (K_(3.0) * xx - yy);
    B[10] = (SH_C3B * xy) * z;
    B[11] = ((-SH_C3C) * y) * ((K_(4.0) * zz - xx) - yy);
    B[12] = (SH_C3D * z) * ((K_(2.0) * zz - K_(3.0) * xx) - K_(3.0) * yy);
    B[13] = ((-SH_C3C) * x) * ((K_(4.0) * zz - xx) - yy);
    B[14] = (SH_C3E * z) * (xx - yy);
    B[15] = ((-SH_C3A) * x) * (xx - K_(3.0) * yy);
}
void orc_sh_basis(const real* d, real* B) { sh_basis(d, B); }

/* Gradient of each basis function w.r.t. the (unconstrained) direction components. */
static void sh_basis_grad(const real* d, real dB[16][3]) {
    real x = d[0], y = d[1], z = d[2];
    real xx = x * x, yy = y * y, zz = z * z;
    memset(dB, 0, sizeof(real) * 48);
    dB[1][1] = -SH_C1;
    dB[2][2] = SH_C1;
    dB[3][0] = -SH_C1;
    dB[4][0] = SH_C2A * y; dB[4][1] = SH_C2A * x;
    dB[5][1] = -SH_C2A * z; dB[5][2] = -SH_C2A * y;
    dB[6][0] = -K_(2.0) * SH_C2B * x; dB[6][1] = -K_(2.0) * SH_C2B * y; dB[6][2] = K_(4.0) * SH_C2B * z;
    dB[7][0] = -SH_C2A * z; dB[7][2] = -SH_C2A * x;
    dB[8][0] = K_(2.0) * SH_C2C * x; dB[8][1] = -K_(2.0) * SH_C2C * y;
    /* B9 = -C3a (3 x^2 y - y^3) */
    dB[9][0] = -SH_C3A * K_(6.0) * x * y; dB[9][1] = -SH_C3A * (K_(3.0) * xx - K_(3.0) * yy);
    /* B10 = C3b x y z */
    dB[10][0] = SH_C3B * y * z; dB[10][1] = SH_C3B * x * z; dB[10][2] = SH_C3B * x * y;
    /* B11 = -C3c (4 y z^2 - x^2 y - y^3) */
    dB[11][0] = SH_C3C * K_(2.0) * x * y; dB[11][1] = -SH_C3C * (K_(4.0) * zz - xx - K_(3.0) * yy);
    dB[11][2] = -SH_C3C * K_(8.0) * y * z;
    /* B12 = C3d (2 z^3 - 3 x^2 z - 3 y^2 z) */
    dB[12][0] = -SH_C3D * K_(6.0) * x * z; dB[12][1] = -SH_C3D * K_(6.0) * y * z;
    dB[12][2] = SH_C3D * (K_(6.0) * zz - K_(3.0) * xx - K_(3.0) * yy);
    /* B13 = -C3c (4 x z^2 - x^3 - x y^2) */
    dB[13][0] = -SH_C3C * (K_(4.0) * zz - K_(3.0) * xx - yy); dB[13][1] = SH_C3C * K_(2.0) * x * y;
    dB[13][2] = -SH_C3C * K_(8.0) * x * z;
    /* B14 = C3e (x^2 z - y^2 z) */
    dB[14][0] = SH_C3E * K_(2.0) * x * z; dB[14][1] = -SH_C3E * K_(2.0) * y * z; dB[14][2] = SH_C3E * (xx - yy);
    /* B15 = -C3a (x^3 - 3 x y^2) */
    dB[15][0] = -SH_C3A * (K_(3.0) * xx - K_(3.0) * yy); dB[15][1] = SH_C3A * K_(6.0) * x * y;
}

/* Intermediates of the projection that both O1 and O6 need. */
typedef struct {
    real t[3];        /* camera-space centre */
    real limx, limy;  /* Jacobian clamp limits */
    real txtz, tytz;  /* unclamped ratios */
    int clx, cly;     /* -1/0/+1: which side the clamp is active on */
    real J00, J02, J11, J12;
    real Tm[6];       /* J * Rcw, 2x3 */
    real Sg[9], Rq[9];
    real a, b, c, det;
} proj_t;

/* O1.1 - O1.4.  Returns 0 if the Gaussian is culled by the near plane. */
static int project(const orc_cam* cam, const real* mu, const real* s, const real* q, proj_t* p) {
    const real* W = cam->Rcw;
    for (int r = 0; r < 3; ++r)
        p->t[r] = ((W[3 * r + 0] * mu[0] + W[3 * r + 1] * mu[1]) + W[3 * r + 2] * mu[2]) + cam->tau[r];
    if (!(p->t[2] > cam->znear)) return 0;
    real tz = p->t[2];
    p->limx = JCLAMP * ((K_(0.5) * (real)cam->W) / cam->fx);
    p->limy = JCLAMP * ((K_(0.5) * (real)cam->H) / cam->fy);
    p->txtz = p->t[0] / tz;
    p->tytz = p->t[1] / tz;
    real cxr = p->txtz, cyr = p->tytz;
    p->clx = 0; p->cly = 0;
    if (cxr > p->limx) { cxr = p->limx; p->clx = 1; } else if (cxr < -p->limx) { cxr = -p->limx; p->clx = -1; }
    if (cyr > p->limy) { cyr = p->limy; p->cly = 1; } else if (cyr < -p->limy) { cyr = -p->limy; p->cly = -1; }
    real txc = cxr * tz, tyc = cyr * tz;
    real tz2 = tz * tz;
    p->J00 = cam->fx / tz;
    p->J02 = -(cam->fx * txc) / tz2;
    p->J11 = cam->fy / tz;
    p->J12 = -(cam->fy * tyc) / tz2;
    for (int c = 0; c < 3; ++c) {
        p->Tm[c] = p->J00 * W[c] + p->J02 * W[6 + c];
        p->Tm[3 + c] = p->J11 * W[3 + c] + p->J12 * W[6 + c];
    }
    cov3d(s, q, p->Sg, p->Rq);
    real V[6];
    for (int r = 0; r < 2; ++r)
        for (int c = 0; c < 3; ++c)
            V[3 * r + c] = p->Tm[3 * r + 0] * p->Sg[c] + p->Tm[3 * r + 1] * p->Sg[3 + c] + p->Tm[3 * r + 2] * p->Sg[6 + c];
    real c00 = V[0] * p->Tm[0] + V[1] * p->Tm[1] + V[2] * p->Tm[2];
    real c01 = V[0] * p->Tm[3] + V[1] * p->Tm[4] + V[2] * p->Tm[5];
    real c11 = V[3] * p->Tm[3] + V[4] * p->Tm[4] + V[5] * p->Tm[5];
    p->a = c00 + LOWPASS;
    p->b = c01;
    p->c = c11 + LOWPASS;
    p->det = p->a * p->c - p->b * p->b;
    return 1;
}

/* camera centre in world space: o_cam = -Rcw^T tau */
static void cam_origin(const orc_cam* cam, real o[3]) {
    const real* W = cam->Rcw;
    for (int c = 0; c < 3; ++c)
        o[c] = -((W[c] * cam->tau[0] + W[3 + c] * cam->tau[1]) + W[6 + c] * cam->tau[2]);
}

/* O1: per-Gaussian projection.  radius == 0 <=> culled (then every other output is 0). */
void orc_preprocess(const orc_cam* cam, int N, int D, const real* mu, const real* sc, const real* qt,
                    const real* op, const real* sh, real* mean2D, real* depth, real* conic_o,
                    real* rgb, int32_t* radius, int32_t* rect, uint32_t* touched, uint8_t* clamped) {
    const int K = (D + 1) * (D + 1);
    const int gx = (cam->W + TILE - 1) / TILE, gy = (cam->H + TILE - 1) / TILE;
    real ocam[3];
    cam_origin(cam, ocam);
    for (int i = 0; i < N; ++i) {
        mean2D[2 * i] = mean2D[2 * i + 1] = 0; depth[i] = 0;
        conic_o[4 * i] = conic_o[4 * i + 1] = conic_o[4 * i + 2] = conic_o[4 * i + 3] = 0;
        rgb[3 * i] = rgb[3 * i + 1] = rgb[3 * i + 2] = 0;
        radius[i] = 0; touched[i] = 0; clamped[i] = 0;
        rect[4 * i] = rect[4 * i + 1] = rect[4 * i + 2] = rect[4 * i + 3] = 0;
        proj_t p;
        if (!project(cam, mu + 3 * i, sc + 3 * i, qt + 4 * i, &p)) continue;
        if (!(p.det > 0)) continue;
        real A = p.c / p.det, B = (-p.b) / p.det, C = p.a / p.det;
        real mid = K_(0.5) * (p.a + p.c);
        real lam = mid + rsqrt_(rmax(LAMBDA_GUARD, mid * mid - p.det));
        real rad = rceil(RADIUS_SIGMAS * rsqrt_(lam));
        real mx = (cam->fx * p.txtz + cam->cx) - K_(0.5);
        real my = (cam->fy * p.tytz + cam->cy) - K_(0.5);
        /* tile rect, clamped in floating point before the integer conversion */
        real fgx = (real)gx, fgy = (real)gy;
        int x0 = (int)rmin(rmax(rfloor((mx - rad) / K_(16.0)), K_(0.0)), fgx);
        int x1 = (int)rmin(rmax(rfloor(((mx + rad) + K_(15.0)) / K_(16.0)), K_(0.0)), fgx);
        int y0 = (int)rmin(rmax(rfloor((my - rad) / K_(16.0)), K_(0.0)), fgy);
        int y1 = (int)rmin(rmax(rfloor(((my + rad) + K_(15.0)) / K_(16.0)), K_(0.0)), fgy);
        int64_t nt = (int64_t)(x1 - x0) * (int64_t)(y1 - y0);
        if (nt <= 0) continue;
        /* colour */
        real v[3] = {mu[3 * i] - ocam[0], mu[3 * i + 1] - ocam[1], mu[3 * i + 2] - ocam[2]};
        real len = rsqrt_((v[0] * v[0] + v[1] * v[1]) + v[2] * v[2]);
        real d[3] = {v[0] / len, v[1] / len, v[2] / len};
        real Bk[16];
        sh_basis(d, Bk);
        uint8_t cl = 0;
        for (int ch = 0; ch < 3; ++ch) {
            const real* s_i = sh + (size_t)i * K * 3;
            real acc = Bk[0] * s_i[ch];
            for (int k = 1; k < K; ++k) acc = acc + Bk[k] * s_i[3 * k + ch];
            acc = acc + K_(0.5);
            if (acc < 0) { acc = 0; cl |= (uint8_t)(1u << ch); }
            rgb[3 * i + ch] = acc;
        }
        mean2D[2 * i] = mx; mean2D[2 * i + 1] = my;
        depth[i] = p.t[2];
        conic_o[4 * i] = A; conic_o[4 * i + 1] = B; conic_o[4 * i + 2] = C; conic_o[4 * i + 3] = op[i];
        radius[i] = (int32_t)rad;
        rect[4 * i] = x0; rect[4 * i + 1] = y0; rect[4 * i + 2] = x1; rect[4 * i + 3] = y1;
        touched[i] = (uint32_t)nt;
        clamped[i] = cl;
    }
}

/* ---------------------------------------------------------------------------------- */
/* O2: binning.  The sorted list is the list of all (tile, Gaussian) pairs ordered by   */
/* (tile_id, depth bits, gaussian id).                                                  */
typedef struct { uint64_t key; uint32_t gid; } pair_t;
static int pair_cmp(const void* a, const void* b) {
    const pair_t* x = (const pair_t*)a; const pair_t* y = (const pair_t*)b;
    if (x->key != y->key) return x->key < y->key ? -1 : 1;
    if (x->gid != y->gid) return x->gid < y->gid ? -1 : 1;
    return 0;
}
static uint32_t depth_bits(real z) { float f = (float)z; uint32_t u; memcpy(&u, &f, 4); return u; }

/* keys/gid have room for sum(touched) pairs; tile_offsets has T+1 entries. Returns P, the number
 * of pairs emitted.  tile_select (nullable, [T]): when given, only pairs whose tile has
 * tile_select[t] != 0 are emitted and every other tile gets an empty range -- the sparse step
 * never reads the ranges of tiles it does not sample (reading R14). */
int64_t orc_bin_sort(const orc_cam* cam, int N, const real* depth, const int32_t* rect,
                     const uint32_t* touched, const uint32_t* tile_select, uint64_t* keys, uint32_t* gid,
                     uint32_t* tile_offsets) {
    const int gx = (cam->W + TILE - 1) / TILE, gy = (cam->H + TILE - 1) / TILE;
    const int T = gx * gy;
    int64_t cap = 0;
    for (int i = 0; i < N; ++i) cap += touched[i];
    pair_t* pr = (pair_t*)malloc(sizeof(pair_t) * (size_t)(cap > 0 ? cap : 1));
    int64_t P = 0;
    for (int i = 0; i < N; ++i) {
        if (!touched[i]) continue;
        uint64_t db = depth_bits(depth[i]);
        for (int ty = rect[4 * i + 1]; ty < rect[4 * i + 3]; ++ty)
            for (int tx = rect[4 * i]; tx < rect[4 * i + 2]; ++tx) {
                const uint32_t t = (uint32_t)(ty * gx + tx);
                if (tile_select && !tile_select[t]) continue;
                pr[P].key = ((uint64_t)t << 32) | db;
                pr[P].gid = (uint32_t)i;
                ++P;
            }
    }
    qsort(pr, (size_t)P, sizeof(pair_t), pair_cmp);
    for (int64_t j = 0; j < P; ++j) { keys[j] = pr[j].key; gid[j] = pr[j].gid; }
    /* tile_offsets[t] = number of pairs with tile_id < t */
    int64_t j = 0;
    for (int t = 0; t <= T; ++t) {
        while (j < P && (int64_t)(pr[j].key >> 32) < t) ++j;
        tile_offsets[t] = (uint32_t)j;
    }
    free(pr);
    return P;
}

/* ---------------------------------------------------------------------------------- */
/* O3: sampling.                                                                        */
static uint64_t mix64(uint64_t seed, uint64_t idx) {
    uint64_t z = seed + (idx + 1ull) * 0x9E3779B97F4A7C15ull;
    z ^= z >> 30; z *= 0xBF58476D1CE4E5B9ull;
    z ^= z >> 27; z *= 0x94D049BB133111EBull;
    z ^= z >> 31;
    return z;
}
uint64_t orc_mix64(uint64_t seed, uint64_t idx) { return mix64(seed, idx); }

/* fixed-point error of one pixel: q = trunc(clamp(e, 0, 15.999) * 2^20), NaN -> 0 */
static uint32_t quant_err(real e) {
    if (!(e > 0)) return 0;
    if (e > ERR_CLAMP) e = ERR_CLAMP;
    return (uint32_t)(e * ERR_SCALE);
}

typedef struct { uint64_t score; uint32_t tile; } ts_t;
static int ts_cmp(const void* a, const void* b) {
    const ts_t* x = (const ts_t*)a; const ts_t* y = (const ts_t*)b;
    if (x->score != y->score) return x->score > y->score ? -1 : 1; /* score descending */
    if (x->tile != y->tile) return x->tile < y->tile ? -1 : 1;      /* tile ascending   */
    return 0;
}
static int u32_cmp(const void* a, const void* b) {
    uint32_t x = *(const uint32_t*)a, y = *(const uint32_t*)b;
    return x < y ? -1 : (x > y ? 1 : 0);
}

/* err == NULL -> e(p) = sum_ch |render - target| (Eq. 2).
 * Outputs: qerr[H*W] (the fixed-point copy), tile_score[T], tiles[k] ascending,
 * tile_pix_offsets[k+1], pix[n] (global y*W+x, tile order, ascending local index).
 * kn[0] = k, kn[1] = n. */
void orc_sample(const orc_cam* cam, const real* err, const real* render, const real* target,
                int pct_num, int pct_den, int pixel_mode, int rate_num, int rate_den, uint64_t seed,
                uint32_t* qerr, uint64_t* tile_score, uint32_t* tiles, uint32_t* tile_pix_offsets,
                uint32_t* pix, int32_t* kn) {
    const int W = cam->W, H = cam->H;
    const int gx = (W + TILE - 1) / TILE, gy = (H + TILE - 1) / TILE, T = gx * gy;
    for (int y = 0; y < H; ++y)
        for (int x = 0; x < W; ++x) {
            size_t p = (size_t)y * W + x;
            real e;
            if (err) e = err[p];
            else e = (rabs(render[3 * p] - target[3 * p]) + rabs(render[3 * p + 1] - target[3 * p + 1])) +
                     rabs(render[3 * p + 2] - target[3 * p + 2]);
            qerr[p] = quant_err(e);
        }
    ts_t* ts = (ts_t*)malloc(sizeof(ts_t) * (size_t)T);
    for (int t = 0; t < T; ++t) {
        int tx = t % gx, ty = t / gx;
        uint64_t sum = 0, cnt = 0;
        for (int ly = 0; ly < TILE; ++ly)
            for (int lx = 0; lx < TILE; ++lx) {
                int x = tx * TILE + lx, y = ty * TILE + ly;
                if (x < W && y < H) { sum += qerr[(size_t)y * W + x]; ++cnt; }
            }
        tile_score[t] = (sum << 8) / cnt; /* fixed-point mean; cnt >= 1 by construction of the grid */
        ts[t].score = tile_score[t]; ts[t].tile = (uint32_t)t;
    }
    int k = (int)(((int64_t)pct_num * T) / pct_den);
    if (k < 1) k = 1;
    if (k > T) k = T;
    qsort(ts, (size_t)T, sizeof(ts_t), ts_cmp);
    for (int i = 0; i < k; ++i) tiles[i] = ts[i].tile;
    qsort(tiles, (size_t)k, sizeof(uint32_t), u32_cmp);
    free(ts);
    uint32_t n = 0;
    for (int i = 0; i < k; ++i) {
        int t = (int)tiles[i], tx = t % gx, ty = t / gx;
        tile_pix_offsets[i] = n;
        uint64_t cnt = 0, S = 0;
        uint32_t qmax = 0; int have = 0; uint32_t pmax = 0;
        for (int ly = 0; ly < TILE; ++ly)
            for (int lx = 0; lx < TILE; ++lx) {
                int x = tx * TILE + lx, y = ty * TILE + ly;
                if (x < W && y < H) {
                    uint32_t q = qerr[(size_t)y * W + x];
                    ++cnt; S += (q >> 8);
                    if (!have || q > qmax) { have = 1; qmax = q; pmax = (uint32_t)((size_t)y * W + x); }
                }
            }
        uint32_t n0 = n;
        for (int ly = 0; ly < TILE; ++ly)
            for (int lx = 0; lx < TILE; ++lx) {
                int x = tx * TILE + lx, y = ty * TILE + ly;
                if (!(x < W && y < H)) continue;
                uint32_t p = (uint32_t)((size_t)y * W + x);
                int keep;
                if (pixel_mode == 0) keep = 1;
                else {
                    uint64_t u16 = mix64(seed, p) >> 48;
                    uint64_t q16 = qerr[p] >> 8;
                    keep = (u16 * S * (uint64_t)rate_den) < ((uint64_t)rate_num * cnt * q16 * 65536ull);
                }
                if (keep) pix[n++] = p;
            }
        if (n == n0) pix[n++] = pmax; /* N_pix >= 1 */
    }
    tile_pix_offsets[k] = n;
    kn[0] = k; kn[1] = (int32_t)n;
}

/* ---------------------------------------------------------------------------------- */
/* O4: sparse forward.  power uses ONE fixed fused sequence so that the fp32 build is a  */
/* bit-level referee for the skip decisions.          */
static real splat_power(real A, real B, real C, real dx, real dy) {
    /* -1/2 (A dx^2 + C dy^2) - B dx dy  ==  ((-B) dy + (-A/2) dx) dx + ((-C/2) dy) dy */
    real nA = K_(-0.5) * A, nB = -B, nC = K_(-0.5) * C;
    return rfma(rfma(nB, dy, nA * dx), dx, (nC * dy) * dy);
}

static real rel_margin(real v, real thr) { return rabs(v - thr) / thr; }

void orc_raster_fwd(const orc_cam* cam, const uint32_t* tile_offsets, const uint32_t* gid_sorted,
                    const real* mean2D, const real* conic_o, const real* rgb, int k,
                    const uint32_t* tiles, const uint32_t* tile_pix_offsets, const uint32_t* pix,
                    real* out_color, real* out_T, uint32_t* n_contrib, uint32_t* n_walked,
                    real* margin /* [n,2]: forward, backward; nullable */,
                    real margin_thr, real* flip_w /* [n]; nullable */) {
    const int W = cam->W;
    for (int it = 0; it < k; ++it) {
        uint32_t t = tiles[it];
        uint32_t start = tile_offsets[t], end = tile_offsets[t + 1];
        for (uint32_t ip = tile_pix_offsets[it]; ip < tile_pix_offsets[it + 1]; ++ip) {
            real px = (real)(pix[ip] % (uint32_t)W), py = (real)(pix[ip] / (uint32_t)W);
            real T = K_(1.0), C[3] = {0, 0, 0};
            uint32_t last = 0, walked = 0;
            real mg = K_(1.0), mgb = K_(1.0); /* distance to the nearest decision threshold */
            /* flip_w: compositing weight that moves if every decision within margin_thr of its threshold is
             * taken the other way: a skipped / kept Gaussian at alpha ~ 1/255
             * moves alpha T of weight onto or off itself and as much off or onto everything behind it; a stop
             * taken or not taken moves at most the transmittance T still unspent at that point. */
            real flip = 0;
            for (uint32_t j = start; j < end; ++j) {
                ++walked;
                uint32_t g = gid_sorted[j];
                real dx = mean2D[2 * g] - px, dy = mean2D[2 * g + 1] - py;
                real power = splat_power(conic_o[4 * g], conic_o[4 * g + 1], conic_o[4 * g + 2], dx, dy);
                if (power > 0) continue;
                real oG = conic_o[4 * g + 3] * rexp(power);
                real alpha = rmin(ALPHA_MAX, oG);
                mg = rmin(mg, rel_margin(oG, ALPHA_MIN));
                if (rel_margin(oG, ALPHA_MIN) < margin_thr) flip += alpha * T;
                if (alpha < ALPHA_MIN) continue;
                mgb = rmin(mgb, rel_margin(oG, ALPHA_MAX)); /* only the derivative jumps at the 0.99 clamp */
                real Tn = T * (K_(1.0) - alpha);
                mg = rmin(mg, rel_margin(Tn, T_MIN));
                if (rel_margin(Tn, T_MIN) < margin_thr) flip += T;
                if (Tn < T_MIN) break;
                real w = alpha * T;
                C[0] += rgb[3 * g] * w; C[1] += rgb[3 * g + 1] * w; C[2] += rgb[3 * g + 2] * w;
                T = Tn;
                last = j - start + 1;
            }
            out_color[3 * ip] = C[0] + T * cam->bg[0];
            out_color[3 * ip + 1] = C[1] + T * cam->bg[1];
            out_color[3 * ip + 2] = C[2] + T * cam->bg[2];
            out_T[ip] = T;
            n_contrib[ip] = last;
            if (n_walked) n_walked[ip] = walked;
            if (margin) { margin[2 * ip] = mg; margin[2 * ip + 1] = rmin(mg, mgb); }
            if (flip_w) flip_w[ip] = flip;
        }
    }
}

/* O5: sparse backward, raster part.  Accumulators are double in both builds. */
void orc_raster_bwd(const orc_cam* cam, int N, const uint32_t* tile_offsets, const uint32_t* gid_sorted,
                    const real* mean2D, const real* conic_o, const real* rgb, int k,
                    const uint32_t* tiles, const uint32_t* tile_pix_offsets, const uint32_t* pix,
                    const real* out_T, const uint32_t* n_contrib, const real* dL_dcolor,
                    real* dL_dmean2D, real* dL_dconic, real* dL_dopac, real* dL_drgb,
                    double* sum_abs /* [N,9] nullable: per gradient element, the sum of |term| over the
                                       (pixel, Gaussian) terms that were added -- the scale fp32 summation-order
                                       noise is measured against; order mean2D[2],
                                       conic[3], opacity, rgb[3] */) {
    const int W = cam->W;
    double* acc = (double*)calloc((size_t)N * 9, sizeof(double));
    if (sum_abs) memset(sum_abs, 0, sizeof(double) * (size_t)N * 9);
    for (int it = 0; it < k; ++it) {
        uint32_t t = tiles[it];
        uint32_t start = tile_offsets[t];
        for (uint32_t ip = tile_pix_offsets[it]; ip < tile_pix_offsets[it + 1]; ++ip) {
            real px = (real)(pix[ip] % (uint32_t)W), py = (real)(pix[ip] / (uint32_t)W);
            const real* g3 = dL_dcolor + 3 * ip;
            real Tf = out_T[ip];
            real T = Tf;
            real S[3] = {0, 0, 0};
            for (uint32_t jj = n_contrib[ip]; jj > 0; --jj) {
                uint32_t j = start + jj - 1;
                uint32_t g = gid_sorted[j];
                real A = conic_o[4 * g], B = conic_o[4 * g + 1], Cc = conic_o[4 * g + 2], o = conic_o[4 * g + 3];
                real dx = mean2D[2 * g] - px, dy = mean2D[2 * g + 1] - py;
                real power = splat_power(A, B, Cc, dx, dy);
                if (power > 0) continue;
                real G = rexp(power);
                real oG = o * G;
                real alpha = rmin(ALPHA_MAX, oG);
                if (alpha < ALPHA_MIN) continue;
                real om = K_(1.0) - alpha;
                T = T / om; /* T_k */
                real w = alpha * T;
                double* a = acc + (size_t)g * 9;
                double* sa = sum_abs ? sum_abs + (size_t)g * 9 : NULL;
                real dL_dalpha = 0;
                for (int ch = 0; ch < 3; ++ch) {
                    real c = rgb[3 * g + ch];
                    a[6 + ch] += (double)(w * g3[ch]);
                    if (sa) sa[6 + ch] += fabs((double)(w * g3[ch]));
                    dL_dalpha += ((c - S[ch]) * T - cam->bg[ch] * Tf / om) * g3[ch];
                    S[ch] = alpha * c + om * S[ch];
                }
                if (oG < ALPHA_MAX) { /* derivative is zero through the active 0.99 clamp */
                    real dL_dpower = oG * dL_dalpha;
                    a[5] += (double)(G * dL_dalpha);
                    a[0] += (double)(dL_dpower * (-A * dx - B * dy));
                    a[1] += (double)(dL_dpower * (-Cc * dy - B * dx));
                    a[2] += (double)(K_(-0.5) * dx * dx * dL_dpower);
                    a[3] += (double)(-dx * dy * dL_dpower);
                    a[4] += (double)(K_(-0.5) * dy * dy * dL_dpower);
                    if (sa) {
                        sa[5] += fabs((double)(G * dL_dalpha));
                        sa[0] += fabs((double)(dL_dpower * (-A * dx - B * dy)));
                        sa[1] += fabs((double)(dL_dpower * (-Cc * dy - B * dx)));
                        sa[2] += fabs((double)(K_(-0.5) * dx * dx * dL_dpower));
                        sa[3] += fabs((double)(-dx * dy * dL_dpower));
                        sa[4] += fabs((double)(K_(-0.5) * dy * dy * dL_dpower));
                    }
                }
            }
        }
    }
    for (int i = 0; i < N; ++i) {
        const double* a = acc + (size_t)i * 9;
        dL_dmean2D[2 * i] = (real)a[0]; dL_dmean2D[2 * i + 1] = (real)a[1];
        dL_dconic[3 * i] = (real)a[2]; dL_dconic[3 * i + 1] = (real)a[3]; dL_dconic[3 * i + 2] = (real)a[4];
        dL_dopac[i] = (real)a[5];
        dL_drgb[3 * i] = (real)a[6]; dL_drgb[3 * i + 1] = (real)a[7]; dL_drgb[3 * i + 2] = (real)a[8];
    }
    free(acc);
}

/* O6: projection backward (per Gaussian).  Gaussians with radius == 0 get zero gradients. */
void orc_project_bwd(const orc_cam* cam, int N, int D, const real* mu, const real* sc, const real* qt,
                     const real* sh, const int32_t* radius, const uint8_t* clamped,
                     const real* dL_dmean2D, const real* dL_dconic, const real* dL_drgb,
                     real* dL_dmu, real* dL_dsc, real* dL_dq, real* dL_dsh) {
    const int K = (D + 1) * (D + 1);
    const real* W = cam->Rcw;
    real ocam[3];
    cam_origin(cam, ocam);
    for (int i = 0; i < N; ++i) {
        real* gmu = dL_dmu + 3 * i; real* gs = dL_dsc + 3 * i; real* gq = dL_dq + 4 * i;
        real* gsh = dL_dsh + (size_t)i * K * 3;
        gmu[0] = gmu[1] = gmu[2] = 0; gs[0] = gs[1] = gs[2] = 0; gq[0] = gq[1] = gq[2] = gq[3] = 0;
        for (int e = 0; e < 3 * K; ++e) gsh[e] = 0;
        if (radius[i] <= 0) continue;
        proj_t p;
        if (!project(cam, mu + 3 * i, sc + 3 * i, qt + 4 * i, &p)) continue;
        if (!(p.det > 0)) continue;
        const real* s = sc + 3 * i; const real* q = qt + 4 * i;
        real tz = p.t[2], tz2 = tz * tz;
        /* conic (A,B,C) -> cov2D (a,b,c):  H = -M Ghat M,  M = [[A,B],[B,C]], Ghat = [[gA, gB/2],[gB/2, gC]] */
        real A = p.c / p.det, B = -p.b / p.det, C = p.a / p.det;
        real gA = dL_dconic[3 * i], gB = dL_dconic[3 * i + 1], gC = dL_dconic[3 * i + 2];
        real hB = K_(0.5) * gB;
        /* X = Ghat M */
        real X00 = gA * A + hB * B, X01 = gA * B + hB * C, X10 = hB * A + gC * B, X11 = hB * B + gC * C;
        real H00 = -(A * X00 + B * X10), H01 = -(A * X01 + B * X11), H11 = -(B * X01 + C * X11);
        /* symmetric 2x2 Hs with dL = <Hs, dcov2D>: entries (H00, H01; H01, H11); dL/db = 2 H01 */
        const real* Tm = p.Tm;
        /* dL/dSigma = Tm^T Hs Tm */
        real HT[6]; /* Hs * Tm, 2x3 */
        for (int c = 0; c < 3; ++c) {
            HT[c] = H00 * Tm[c] + H01 * Tm[3 + c];
            HT[3 + c] = H01 * Tm[c] + H11 * Tm[3 + c];
        }
        real dSg[9];
        for (int r = 0; r < 3; ++r)
            for (int c = 0; c < 3; ++c) dSg[3 * r + c] = Tm[r] * HT[c] + Tm[3 + r] * HT[3 + c];
        /* dL/dTm = 2 Hs Tm Sigma */
        real dTm[6];
        for (int r = 0; r < 2; ++r)
            for (int c = 0; c < 3; ++c)
                dTm[3 * r + c] = K_(2.0) * (HT[3 * r + 0] * p.Sg[c] + HT[3 * r + 1] * p.Sg[3 + c] + HT[3 * r + 2] * p.Sg[6 + c]);
        /* Tm = J Rcw  =>  dL/dJ = dTm Rcw^T ; only J00, J02, J11, J12 are variables */
        real dJ00 = dTm[0] * W[0] + dTm[1] * W[1] + dTm[2] * W[2];
        real dJ02 = dTm[0] * W[6] + dTm[1] * W[7] + dTm[2] * W[8];
        real dJ11 = dTm[3] * W[3] + dTm[4] * W[4] + dTm[5] * W[5];
        real dJ12 = dTm[3] * W[6] + dTm[4] * W[7] + dTm[5] * W[8];
        real gmx = dL_dmean2D[2 * i], gmy = dL_dmean2D[2 * i + 1];
        real dt[3] = {0, 0, 0};
        /* J00 = fx/tz, J11 = fy/tz */
        dt[2] += -(cam->fx / tz2) * dJ00 - (cam->fy / tz2) * dJ11;
        /* J02 = -fx tx~/tz^2 with tx~ = tx (unclamped) or +-lim tz (clamped) */
        if (p.clx == 0) { dt[0] += -(cam->fx / tz2) * dJ02; dt[2] += (K_(2.0) * cam->fx * p.t[0] / (tz2 * tz)) * dJ02; }
        else dt[2] += ((real)p.clx * cam->fx * p.limx / tz2) * dJ02;
        if (p.cly == 0) { dt[1] += -(cam->fy / tz2) * dJ12; dt[2] += (K_(2.0) * cam->fy * p.t[1] / (tz2 * tz)) * dJ12; }
        else dt[2] += ((real)p.cly * cam->fy * p.limy / tz2) * dJ12;
        /* mean2D = f t_xy / tz + c - 0.5 (unclamped t) */
        dt[0] += gmx * cam->fx / tz;
        dt[1] += gmy * cam->fy / tz;
        dt[2] += -gmx * cam->fx * p.t[0] / tz2 - gmy * cam->fy * p.t[1] / tz2;
        /* t = Rcw mu + tau */
        for (int c = 0; c < 3; ++c) gmu[c] = W[c] * dt[0] + W[3 + c] * dt[1] + W[6 + c] * dt[2];
        /* Sigma = M M^T, M = R diag(s): dL/dM = 2 dSg M (dSg symmetric) */
        const real* R = p.Rq;
        real M[9], dM[9];
        for (int r = 0; r < 3; ++r)
            for (int c = 0; c < 3; ++c) M[3 * r + c] = R[3 * r + c] * s[c];
        for (int r = 0; r < 3; ++r)
            for (int c = 0; c < 3; ++c)
                dM[3 * r + c] = K_(2.0) * (dSg[3 * r + 0] * M[c] + dSg[3 * r + 1] * M[3 + c] + dSg[3 * r + 2] * M[6 + c]);
        for (int c = 0; c < 3; ++c) gs[c] = R[c] * dM[c] + R[3 + c] * dM[3 + c] + R[6 + c] * dM[6 + c];
        real dR[9]; /* R' = dM diag(s) */
        for (int r = 0; r < 3; ++r)
            for (int c = 0; c < 3; ++c) dR[3 * r + c] = dM[3 * r + c] * s[c];
        real w = q[0], x = q[1], y = q[2], z = q[3];
        gq[0] = K_(2.0) * (z * (dR[3] - dR[1]) + y * (dR[2] - dR[6]) + x * (dR[7] - dR[5]));
        gq[1] = K_(2.0) * (y * (dR[1] + dR[3]) + z * (dR[2] + dR[6]) + w * (dR[7] - dR[5])) - K_(4.0) * x * (dR[4] + dR[8]);
        gq[2] = K_(2.0) * (x * (dR[1] + dR[3]) + w * (dR[2] - dR[6]) + z * (dR[5] + dR[7])) - K_(4.0) * y * (dR[0] + dR[8]);
        gq[3] = K_(2.0) * (w * (dR[3] - dR[1]) + x * (dR[2] + dR[6]) + y * (dR[5] + dR[7])) - K_(4.0) * z * (dR[0] + dR[4]);
        /* colour: rgb_ch = max(0, 0.5 + sum_k B_k(d) sh[k][ch]) */
        real v[3] = {mu[3 * i] - ocam[0], mu[3 * i + 1] - ocam[1], mu[3 * i + 2] - ocam[2]};
        real len = rsqrt_((v[0] * v[0] + v[1] * v[1]) + v[2] * v[2]);
        real d[3] = {v[0] / len, v[1] / len, v[2] / len};
        real Bk[16], dB[16][3];
        sh_basis(d, Bk);
        sh_basis_grad(d, dB);
        real dd[3] = {0, 0, 0};
        const real* s_i = sh + (size_t)i * K * 3;
        for (int ch = 0; ch < 3; ++ch) {
            if (clamped[i] & (1u << ch)) continue;
            real g = dL_drgb[3 * i + ch];
            for (int kk = 0; kk < K; ++kk) {
                gsh[3 * kk + ch] = Bk[kk] * g;
                for (int c = 0; c < 3; ++c) dd[c] += dB[kk][c] * s_i[3 * kk + ch] * g;
            }
        }
        /* d = v/|v|: dL/dv = (dd - d (d . dd)) / |v| */
        real dot = d[0] * dd[0] + d[1] * dd[1] + d[2] * dd[2];
        for (int c = 0; c < 3; ++c) gmu[c] += (dd[c] - d[c] * dot) / len;
    }
}

/* Dense reference render used by the "full mask == dense" pin: a plain per-pixel loop over the
 * whole image, written independently of the CSR pixel-list machinery of orc_raster_fwd. */
void orc_render_dense(const orc_cam* cam, const uint32_t* tile_offsets, const uint32_t* gid_sorted,
                      const real* mean2D, const real* conic_o, const real* rgb, real* image /*[H,W,3]*/) {
    const int W = cam->W, H = cam->H, gx = (W + TILE - 1) / TILE;
    for (int y = 0; y < H; ++y)
        for (int x = 0; x < W; ++x) {
            int t = (y / TILE) * gx + (x / TILE);
            real T = K_(1.0), C[3] = {0, 0, 0};
            for (uint32_t j = tile_offsets[t]; j < tile_offsets[t + 1]; ++j) {
                uint32_t g = gid_sorted[j];
                real dx = mean2D[2 * g] - (real)x, dy = mean2D[2 * g + 1] - (real)y;
                real power = splat_power(conic_o[4 * g], conic_o[4 * g + 1], conic_o[4 * g + 2], dx, dy);
                if (power > 0) continue;
                real alpha = rmin(ALPHA_MAX, conic_o[4 * g + 3] * rexp(power));
                if (alpha < ALPHA_MIN) continue;
                real Tn = T * (K_(1.0) - alpha);
                if (Tn < T_MIN) break;
                real w = alpha * T;
                C[0] += rgb[3 * g] * w; C[1] += rgb[3 * g + 1] * w; C[2] += rgb[3 * g + 2] * w;
                T = Tn;
            }
            size_t p = (size_t)y * W + x;
            image[3 * p] = C[0] + T * cam->bg[0];
            image[3 * p + 1] = C[1] + T * cam->bg[1];
            image[3 * p + 2] = C[2] + T * cam->bg[2];
        }
}

/* O7 orc_loss_sparse: sparse supervision on the sampled pixels.
 *   PAPER.md:168-208 Sec. 3.7 Eq. 9-11, Eq. 17-18.  Readings (R19-R23):
 *   - pixel term: Charbonnier l1(p) = 1/3 sum_c sqrt((x_c - y_c)^2 + eps_l1^2)   (Eq. 17 left is its derivative)
 *   - tile term (Eq. 9): per colour channel, over the tile's m sampled pixels, population statistics
 *       NCC_c = cov_xy / sqrt(var_x var_y + eps_ncc),   L_ncc^tau = 1/3 sum_c (1 - NCC_c)
 *     with the per-pixel gradient of Eq. 17 right (exact derivative of m L_ncc^tau, eps placed as written here):
 *       gN_{p,c} = m dL_ncc/dx_{p,c} = -1/3 [ (y - mu_y)/sqrt(var_x var_y + eps) - NCC_c var_y (x - mu_x)/(var_x var_y + eps) ]
 *   - Eq. 10: gbar_k = mean over the tile's pixels of the 1-norm (over channels) of the per-pixel gradient of
 *     term k (dl1/dx and gN); lambda = clip(gbar_l1 / (gbar_ncc + eps_lam), 0, 1), a constant for the derivative
 *   - Eq. 11 / 18: every sampled pixel carries its tile's term (the expectation over tiles is pixel weighted,
 *     which is what makes the per-pixel gradients of Eq. 17-18, printed without 1/m, the exact derivative):
 *       L = 1/n sum_p [ l1(p) + lambda_tau(p) L_ncc^tau(p) ],   dL/dx_{p,c} = 1/n (dl1/dx + lambda gN)
 *     (the minus sign in front of lambda in Eq. 18 contradicts Eq. 11 and Eq. 17; Eq. 11 decides)
 *   - pix_err(p) = sum_c |x_c - y_c|  (Eq. 2), the per-pixel error the error map is updated with
 * tile_stats[k,3] = { sum_p l1(p), L_ncc^tau, lambda_tau };  loss[2] = { 1/n sum_p l1, 1/n sum_tau lambda m L_ncc }. */
void orc_loss_sparse(const orc_cam* cam, int k, const uint32_t* tpo, const uint32_t* pix, const real* color,
                     const real* target, real eps_l1, real eps_ncc, real eps_lam, real* dL_dcolor, real* pix_err,
                     real* tile_stats, real* loss) {
    (void)cam;
    const uint32_t n = tpo[k];
    real L1 = 0, LN = 0;
    for (int it = 0; it < k; ++it) {
        const uint32_t p0 = tpo[it], m = tpo[it + 1] - p0;
        real l1sum = 0, g1bar = 0, Lncc = 0, gNbar = 0;
        /* pixel term and its gradient (stored unscaled in dL_dcolor for now) */
        for (uint32_t i = 0; i < m; ++i) {
            const uint32_t s = p0 + i, id = pix[s];
            real e = 0, l = 0;
            for (int c = 0; c < 3; ++c) {
                real d = color[3 * s + c] - target[3 * (size_t)id + c];
                real ch = rsqrt_(d * d + eps_l1 * eps_l1);
                l += ch;
                e += rabs(d);
                dL_dcolor[3 * s + c] = (d / ch) / K_(3.0);
                g1bar += rabs((d / ch) / K_(3.0));
            }
            l1sum += l / K_(3.0);
            pix_err[s] = e;
        }
        /* tile term: statistics per channel, then the gradient; gN kept in a scratch pass */
        real mu_x[3], mu_y[3], vx[3], vy[3], cxy[3], ncc[3], den[3];
        for (int c = 0; c < 3; ++c) {
            real sx = 0, sy = 0;
            for (uint32_t i = 0; i < m; ++i) { sx += color[3 * (p0 + i) + c]; sy += target[3 * (size_t)pix[p0 + i] + c]; }
            mu_x[c] = m ? sx / (real)m : 0; mu_y[c] = m ? sy / (real)m : 0;
            real a = 0, b = 0, ab = 0;
            for (uint32_t i = 0; i < m; ++i) {
                real dx = color[3 * (p0 + i) + c] - mu_x[c], dy = target[3 * (size_t)pix[p0 + i] + c] - mu_y[c];
                a += dx * dx; b += dy * dy; ab += dx * dy;
            }
            vx[c] = m ? a / (real)m : 0; vy[c] = m ? b / (real)m : 0; cxy[c] = m ? ab / (real)m : 0;
            den[c] = vx[c] * vy[c] + eps_ncc;
            ncc[c] = cxy[c] / rsqrt_(den[c]);
            Lncc += (K_(1.0) - ncc[c]) / K_(3.0);
        }
        for (uint32_t i = 0; i < m; ++i)
            for (int c = 0; c < 3; ++c) {
                real dx = color[3 * (p0 + i) + c] - mu_x[c], dy = target[3 * (size_t)pix[p0 + i] + c] - mu_y[c];
                real gN = -(dy / rsqrt_(den[c]) - ncc[c] * vy[c] * dx / den[c]) / K_(3.0);
                gNbar += rabs(gN);
            }
        if (m) { g1bar /= (real)m; gNbar /= (real)m; }
        real lam = rmin(K_(1.0), rmax(K_(0.0), g1bar / (gNbar + eps_lam)));
        for (uint32_t i = 0; i < m; ++i)
            for (int c = 0; c < 3; ++c) {
                real dx = color[3 * (p0 + i) + c] - mu_x[c], dy = target[3 * (size_t)pix[p0 + i] + c] - mu_y[c];
                real gN = -(dy / rsqrt_(den[c]) - ncc[c] * vy[c] * dx / den[c]) / K_(3.0);
                dL_dcolor[3 * (p0 + i) + c] = (dL_dcolor[3 * (p0 + i) + c] + lam * gN) / (real)n;
            }
        tile_stats[3 * it] = l1sum; tile_stats[3 * it + 1] = Lncc; tile_stats[3 * it + 2] = lam;
        L1 += l1sum; LN += lam * (real)m * Lncc;
    }
    loss[0] = n ? L1 / (real)n : 0;
    loss[1] = n ? LN / (real)n : 0;
}

/* O8 orc_raster_stats: statistics forward (Sec. 3.8 Eq. 12,
 * Alg. 1 step 11 "rasterize_forward_pixels").  The same front-to-back walk as O4 (same thresholds, same
 * stopping rule); every composited (pixel, Gaussian) pair with weight w = T alpha adds
 *     E_i += e(p) w,   D_i += D_i(p) w,   W_i += w,
 * where e(p) is the per-pixel error handed in (pix_err[n], sampled-pixel order) and D_i(p) = d^T Sigma'^-1 d
 * = -2 power is the conic Mahalanobis distance between the splat centre and the pixel.
 * stats[N,3] = {E, D, W}; accumulators are double in both builds.  out_depth[n] (nullable) = sum_i w z_i,
 * the expected depth of the sampled pixel (the "depth output" of SURVEY.md f3). */
void orc_raster_stats(const orc_cam* cam, int N, const uint32_t* tile_offsets, const uint32_t* gid_sorted,
                      const real* mean2D, const real* conic_o, const real* depth, int k, const uint32_t* tiles,
                      const uint32_t* tile_pix_offsets, const uint32_t* pix, const real* pix_err, real* stats,
                      real* out_depth) {
    const int W = cam->W;
    double* acc = (double*)calloc((size_t)N * 3, sizeof(double));
    for (int it = 0; it < k; ++it) {
        uint32_t t = tiles[it];
        uint32_t start = tile_offsets[t], end = tile_offsets[t + 1];
        for (uint32_t ip = tile_pix_offsets[it]; ip < tile_pix_offsets[it + 1]; ++ip) {
            real px = (real)(pix[ip] % (uint32_t)W), py = (real)(pix[ip] / (uint32_t)W);
            real T = K_(1.0);
            double z = 0;
            for (uint32_t j = start; j < end; ++j) {
                uint32_t g = gid_sorted[j];
                real dx = mean2D[2 * g] - px, dy = mean2D[2 * g + 1] - py;
                real power = splat_power(conic_o[4 * g], conic_o[4 * g + 1], conic_o[4 * g + 2], dx, dy);
                if (power > 0) continue;
                real alpha = rmin(ALPHA_MAX, conic_o[4 * g + 3] * rexp(power));
                if (alpha < ALPHA_MIN) continue;
                real Tn = T * (K_(1.0) - alpha);
                if (Tn < T_MIN) break;
                real w = alpha * T;
                acc[3 * (size_t)g] += (double)(pix_err[ip] * w);
                acc[3 * (size_t)g + 1] += (double)(K_(-2.0) * power * w);
                acc[3 * (size_t)g + 2] += (double)w;
                z += (double)(w * depth[g]);
                T = Tn;
            }
            if (out_depth) out_depth[ip] = (real)z;
        }
    }
    for (size_t i = 0; i < (size_t)N * 3; ++i) stats[i] = (real)acc[i];
    free(acc);
}

/* O9 orc_sample_paper / orc_maps_update: the paper's own sampler and its persistent maps (SURVEY.md 8f row
 * f2; Eq. 3-4, Sec. 3.5 Eq. 7-8).  Every tile is sampled with
 * N = min(n_pix, #in-image pixels) pixels: n_hard by multinomial sampling WITHOUT replacement from
 * pi_E (Eq. 7), n_stable by TopK of the age map over the rest (Eq. 8), the remainder uniformly without
 * replacement.  Readings (R26-R29), all integer so that both sides agree bit for bit:
 *   - weight of a pixel: q = 1 + trunc(min(E, 15.999) * 2^16) from the fp16 error map (E <= 0 or NaN -> 1): the
 *     "+ eps" of Eq. 7 as one fixed-point unit per pixel, so a tile of zero errors is sampled uniformly
 *   - draw d of tile t: r = mix64(seed, t << 16 | d) mod (sum of the remaining q); the pixel whose running sum
 *     of q in ascending local index first exceeds r is taken and removed (sequential multinomial w/o replacement)
 *   - TopK ties: larger age first, then smaller local index
 *   - remainder draw d: r = mix64(seed ^ 0x5bd1e995a5a5a5a5, t << 16 | d) mod (#remaining): the r-th remaining pixel
 *   - output: tiles = 0..T-1, per tile the chosen pixels in ascending local index (row-major inside the tile). */
static float half_bits_to_float(uint16_t h) { _Float16 x; memcpy(&x, &h, 2); return (float)x; }
static uint16_t float_to_half_bits(float f) { _Float16 x = (_Float16)f; uint16_t h; memcpy(&h, &x, 2); return h; }
uint16_t orc_float_to_half(float f) { return float_to_half_bits(f); }
float orc_half_to_float(uint16_t h) { return half_bits_to_float(h); }

static uint32_t half_weight(uint16_t h) {
    float e = half_bits_to_float(h);
    if (!(e > 0.0f)) return 1u;
    if (e > 15.999f) e = 15.999f;
    return 1u + (uint32_t)(e * 65536.0f);
}

void orc_sample_paper(const orc_cam* cam, const uint16_t* E_half, const uint16_t* age, int n_pix, int n_hard,
                      int n_stable, uint64_t seed, uint32_t* tiles, uint32_t* tpo, uint32_t* pix, int32_t* kn) {
    const int W = cam->W, H = cam->H, gx = (W + TILE - 1) / TILE, gy = (H + TILE - 1) / TILE, T = gx * gy;
    uint32_t n = 0;
    for (int t = 0; t < T; ++t) {
        const int tx = t % gx, ty = t / gx;
        uint32_t q[256], ag[256], id[256];
        int in[256], chosen[256], cnt = 0;
        for (int l = 0; l < 256; ++l) {
            int x = tx * TILE + (l % TILE), y = ty * TILE + (l / TILE);
            in[l] = x < W && y < H;
            chosen[l] = 0;
            if (in[l]) {
                id[l] = (uint32_t)(y * W + x);
                q[l] = half_weight(E_half[id[l]]);
                ag[l] = age[id[l]];
                ++cnt;
            }
        }
        const int N = imin(n_pix, cnt), Nh = imin(n_hard, N), Ns = imin(n_stable, N - Nh), Nr = N - Nh - Ns;
        for (int d = 0; d < Nh; ++d) {                         /* Eq. 7: hard pixels */
            uint64_t S = 0;
            for (int l = 0; l < 256; ++l) if (in[l] && !chosen[l]) S += q[l];
            uint64_t r = mix64(seed, ((uint64_t)t << 16) | (uint64_t)d) % S, acc = 0;
            for (int l = 0; l < 256; ++l) if (in[l] && !chosen[l]) { acc += q[l]; if (r < acc) { chosen[l] = 1; break; } }
        }
        for (int d = 0; d < Ns; ++d) {                         /* Eq. 8: the oldest of the rest */
            int best = -1;
            for (int l = 0; l < 256; ++l) if (in[l] && !chosen[l] && (best < 0 || ag[l] > ag[best])) best = l;
            chosen[best] = 1;
        }
        for (int d = 0; d < Nr; ++d) {                         /* remainder: uniform over what is left */
            uint64_t R = 0;
            for (int l = 0; l < 256; ++l) if (in[l] && !chosen[l]) ++R;
            uint64_t r = mix64(seed ^ 0x5bd1e995a5a5a5a5ull, ((uint64_t)t << 16) | (uint64_t)d) % R, acc = 0;
            for (int l = 0; l < 256; ++l) if (in[l] && !chosen[l]) { if (acc == r) { chosen[l] = 1; break; } ++acc; }
        }
        tiles[t] = (uint32_t)t;
        tpo[t] = n;
        for (int l = 0; l < 256; ++l) if (in[l] && chosen[l]) pix[n++] = id[l];
    }
    tpo[T] = n;
    kn[0] = T; kn[1] = (int32_t)n;
}

/* Eq. 4 then Eq. 3: every age + 1 (saturating at 65535), sampled pixels reset to 0; at the sampled pixels
 * E <- fp16( (1 - beta) * E + beta * e ) with the three operations rounded in fp32 (the paper stores E in half
 * precision; arithmetic precision is this library's: fp32, R0). */
void orc_maps_update(const orc_cam* cam, uint16_t* E_half, uint16_t* age, int n, const uint32_t* pix,
                     const float* pix_err, float beta) {
    const size_t np = (size_t)cam->W * (size_t)cam->H;
    for (size_t p = 0; p < np; ++p) if (age[p] != 0xffffu) ++age[p];
    const float omb = 1.0f - beta;
    for (int i = 0; i < n; ++i) {
        const uint32_t p = pix[i];
        const float a = omb * half_bits_to_float(E_half[p]);
        const float b = beta * pix_err[i];
        E_half[p] = float_to_half_bits(a + b);
        age[p] = 0;
    }
}
