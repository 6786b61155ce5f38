/*
 * soc_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, fp64, single-threaded CPU statement of the per-frequency photon-package
 * simulation of SOC (Juvela, arXiv:1812.06632) and of the energy-balance temperature
 * lookup.  It exists so that the CUDA path can be checked against something that can be
 * read next to the paper.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may load it.  It shares no code, header, table
 * or constant generator with paper_1812_06632_b200/csrc.
 *
 * What the paper fixes (PAPER.md = /root/reference/PAPER.md):
 *   - grid: regular Cartesian root grid of cubic cells, octree refinement into "octets",
 *     one cell vector, root level first then level 2, ...; parent -> first child link,
 *     one reverse link per octet; every cell change is a partial tree traversal, up to
 *     the common parent and down to the new leaf            (Sect. 2.1.1)
 *   - per frequency the kernel sees density, optical depth and an absorption counter;
 *     host loops over frequencies
 *   - absorbed energy integrated over frequency -> temperature, separate kernel;
 *     cells never hit get an ad hoc constant temperature
 *   - sources: isotropic external background, blackbody point sources, a source may sit
 *     in a zero-density cell
 * Everything the paper is silent on (RNG stream, emission sampling, tie-break, free path
 * in scattering optical depth with continuous absorption, Henyey-Greenstein angle,
 * termination, quadrature, table form) follows the readings S1-S16 listed in DESIGN.md
 * (taken from SURVEY.md 8c and BASELINE.json:north_star).
 *
 * Precision (reading S11; north_star "a plain, slow fp64 CPU implementation", SURVEY.md 8c S11 "oracle
 * fp64 throughout"): soc_oracle_simulate -- THE oracle -- holds and evaluates everything in fp64.
 *
 * soc_oracle_simulate_f32state is a second, named entry over the same walk (the same lines of code; the
 * only difference is keep() below): in-cell position, direction and remaining optical depth are rounded
 * to fp32 each time they are stored, every update still being evaluated in fp64.  Why it exists: the walk
 * through a cloud with sharp density contrasts is a chaotic map where packages scatter many times (a
 * lateral shift changes the chord lengths in dense cells, hence where the next scattering falls), so two
 * correct fp64 evaluations that differ in the last bit of a log or a sincos part ways on some packages;
 * on a state snapped to the fp32 lattice they stay together, which is what package-by-package replay of
 * the CUDA path needs at the UV frequencies of configs 3 and 5.  Its licence: tests/test_oracle_pins.py
 * pins it to the fp64 oracle (identical records on non-scattering paths, >= 99 % identical records on
 * config-1/2-like runs, per-cell agreement within 5 sigma of the MC noise over 8 seeds, the same closed
 * forms), and tests/test_gpu_parity.py measures the fp64-state replay match it replaces.  Only the
 * replay-parity tests use it.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): Philox known answers, slab transmission
 * exp(-tau), optically thin bath A = 4 pi I kabs rho V, energy conservation 1e-9,
 * point-source escape fraction by quadrature, HG moments, emission laws / mean number of
 * cells crossed, brute-force geometric replay on tiny octrees, fully-refined == regular
 * 2N identity, temperature power law.  No function here is "parity unpinned".
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define SOC_O_PI 3.14159265358979323846

/* ------------------------------------------------------------------ a1: RNG ---------
 * Philox4x32-10 (Salmon, Moraes, Dror, Shaw 2011), standard multipliers and Weyl
 * constants.  Block b of package p at frequency index f with a 64-bit seed:
 *   counter = (b, p & 0xffffffff, p >> 32, f),  key = (seed & 0xffffffff, seed >> 32)
 * Word -> uniform  u = ((x >> 9) + 0.5) * 2^-23, exactly representable in fp32 and fp64.
 * (north_star: "counter-based Philox4x32 stream per package keyed by (seed, frequency,
 * package id)"; layout = reading S2.) */
void soc_oracle_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        uint64_t p0 = (uint64_t)0xD2511F53u * (uint64_t)c0;
        uint64_t p1 = (uint64_t)0xCD9E8D57u * (uint64_t)c2;
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        uint32_t n1 = (uint32_t)p1;
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        uint32_t n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

void soc_oracle_stream_block(uint64_t seed, int32_t ifreq, int64_t pkg, uint32_t block, uint32_t out[4])
{
    uint32_t ctr[4] = { block, (uint32_t)((uint64_t)pkg & 0xffffffffu), (uint32_t)((uint64_t)pkg >> 32),
                        (uint32_t)ifreq };
    uint32_t key[2] = { (uint32_t)(seed & 0xffffffffu), (uint32_t)(seed >> 32) };
    soc_oracle_philox4x32_10(ctr, key, out);
}

double soc_oracle_uniform(uint32_t word)
{
    return ((double)(word >> 9) + 0.5) * (1.0 / 8388608.0);
}

/* ------------------------------------------------------------------ a8: scattering --
 * Henyey-Greenstein polar angle (north_star; the paper itself tabulates scattering
 * functions).  With mu0 = 2u - 1 the inverse CDF
 *   cos = (1 + g^2 - ((1 - g^2)/(1 - g + 2 g u))^2) / (2 g)
 * is rewritten without the 1/g cancellation (reading S6):
 *   cos = [mu0 + g (3 + mu0^2)/2 + g^2 mu0 + g^3 (mu0^2 - 1)/2] / (1 + g mu0)^2 . */
double soc_oracle_hg_cos(double g, double u)
{
    double mu0 = 2.0 * u - 1.0;
    double num = mu0 + g * (3.0 + mu0 * mu0) * 0.5 + g * g * mu0 + g * g * g * (mu0 * mu0 - 1.0) * 0.5;
    double den = (1.0 + g * mu0) * (1.0 + g * mu0);
    double c = num / den;
    if (c > 1.0) c = 1.0;
    if (c < -1.0) c = -1.0;
    return c;
}

/* New direction at polar angle acos(cost) and azimuth phi about d (reading: rotation
 * basis of Duff et al. 2017, no singular direction), then renormalised. */
void soc_oracle_rotate(const double d[3], double cost, double phi, double out[3])
{
    double sint = sqrt(fmax(0.0, 1.0 - cost * cost));
    double sg = copysign(1.0, d[2]);
    double a = -1.0 / (sg + d[2]);
    double b = d[0] * d[1] * a;
    double t1[3] = { 1.0 + sg * d[0] * d[0] * a, sg * b, -sg * d[0] };
    double t2[3] = { b, sg + d[1] * d[1] * a, -d[1] };
    double cp = cos(phi), sp = sin(phi);
    double n[3];
    for (int j = 0; j < 3; ++j) n[j] = sint * cp * t1[j] + sint * sp * t2[j] + cost * d[j];
    double inv = 1.0 / sqrt(n[0] * n[0] + n[1] * n[1] + n[2] * n[2]);
    for (int j = 0; j < 3; ++j) out[j] = n[j] * inv;
}

/* ------------------------------------------------------------------ grid ------------
 * Cell vector, level-major.  Level l = 1..n_levels has n_cells[l-1] cells,
 * global id = level_off[l-1] + c.  Root index c = ix + nx (iy + ny iz).  For l > 1 the
 * octet is c >> 3 and the slot c & 7 = bx + 2 by + 4 bz.  child[gid] = -1 for a leaf,
 * else the index (within level l+1, a multiple of 8) of the first cell of its octet.
 * parent[l-1][c >> 3] = index (within level l-1) of the parent: one reverse link per
 * octet, as in the paper. */
typedef struct soc_oracle_grid {
    int32_t nx, ny, nz, n_levels;
    int64_t *level_off;   /* [n_levels + 1] */
    int64_t n_total;
    float *rho;           /* [n_total], own copy */
    int32_t *child;       /* [n_total], own copy (all -1 when n_levels == 1) */
    int32_t **parent;     /* [n_levels]; parent[0] = NULL */
} soc_oracle_grid;

void soc_oracle_grid_destroy(soc_oracle_grid *G)
{
    if (!G) return;
    if (G->parent) {
        for (int l = 0; l < G->n_levels; ++l) free(G->parent[l]);
        free(G->parent);
    }
    free(G->level_off); free(G->rho); free(G->child); free(G);
}

/* Returns NULL on an inconsistent hierarchy. */
soc_oracle_grid *soc_oracle_grid_create(int32_t nx, int32_t ny, int32_t nz, int32_t n_levels,
                                        const int64_t *n_cells, const float *rho, const int32_t *child)
{
    if (nx < 1 || ny < 1 || nz < 1 || n_levels < 1) return NULL;
    if (n_cells[0] != (int64_t)nx * ny * nz) return NULL;
    soc_oracle_grid *G = (soc_oracle_grid *)calloc(1, sizeof(*G));
    G->nx = nx; G->ny = ny; G->nz = nz; G->n_levels = n_levels;
    G->level_off = (int64_t *)calloc((size_t)n_levels + 1, sizeof(int64_t));
    for (int l = 0; l < n_levels; ++l) {
        if (l > 0 && (n_cells[l] % 8 != 0)) { soc_oracle_grid_destroy(G); return NULL; }
        G->level_off[l + 1] = G->level_off[l] + n_cells[l];
    }
    G->n_total = G->level_off[n_levels];
    G->rho = (float *)malloc(sizeof(float) * (size_t)G->n_total);
    G->child = (int32_t *)malloc(sizeof(int32_t) * (size_t)G->n_total);
    memcpy(G->rho, rho, sizeof(float) * (size_t)G->n_total);
    if (child) memcpy(G->child, child, sizeof(int32_t) * (size_t)G->n_total);
    else for (int64_t i = 0; i < G->n_total; ++i) G->child[i] = -1;
    G->parent = (int32_t **)calloc((size_t)n_levels, sizeof(int32_t *));
    for (int l = 1; l < n_levels; ++l) {
        int64_t n_oct = n_cells[l] / 8;
        G->parent[l] = (int32_t *)malloc(sizeof(int32_t) * (size_t)(n_oct > 0 ? n_oct : 1));
        for (int64_t o = 0; o < n_oct; ++o) G->parent[l][o] = -1;
    }
    for (int l = 0; l < n_levels; ++l) {
        for (int64_t c = 0; c < n_cells[l]; ++c) {
            int64_t gid = G->level_off[l] + c;
            int32_t ch = G->child[gid];
            if (ch < 0) {
                if (!(G->rho[gid] >= 0.0f) || !isfinite(G->rho[gid])) { soc_oracle_grid_destroy(G); return NULL; }
                continue;
            }
            if (l + 1 >= n_levels || (ch & 7) != 0 || ch + 8 > n_cells[l + 1] ||
                G->parent[l + 1][ch >> 3] != -1) { soc_oracle_grid_destroy(G); return NULL; }
            G->parent[l + 1][ch >> 3] = (int32_t)c;
        }
    }
    for (int l = 1; l < n_levels; ++l)
        for (int64_t o = 0; o < n_cells[l] / 8; ++o)
            if (G->parent[l][o] < 0) { soc_oracle_grid_destroy(G); return NULL; }
    return G;
}

/* ------------------------------------------------------------------ package state --- */
typedef struct {
    int32_t level;      /* l = 1..n_levels */
    int32_t cell;       /* index within the level: authoritative, never re-derived (S4) */
    double f[3];        /* position inside the cell, in units of the cell edge, [0,1]^3 */
    double d[3];        /* unit direction */
    int32_t f32state;   /* 0: the oracle (fp64 throughout); 1: soc_oracle_simulate_f32state, see keep() */
} soc_oracle_state;

/* The value of x as the package state stores it: x itself in the oracle; rounded to fp32 in the
 * f32state variant (header, "Precision").  Everything else is common to both. */
static double keep(double x, int32_t f32state) { return f32state ? (double)(float)x : x; }

typedef struct {
    double bg_intensity;   /* I_nu of the isotropic background, 0 = none */
    int32_t n_point;
    const double *ps_pos;  /* [n_point][3] root-grid units, strictly inside the grid */
    const double *ps_lum;  /* [n_point] */
    int64_t n_bg;          /* ids [0,n_bg) background, the rest point sources; -1 = default split */
    const double *beam;    /* test hook: [6] = position, direction; every package is this beam, E0 = 1 */
    /* f1, dust re-emission: the LAST n_dust package ids are emitted by the cells themselves */
    int64_t n_dust;            /* 0 = none; must equal the sum of dust_count */
    const float *dust_T;       /* [n_total] dust temperature per cell (what soc_oracle_update_temperatures wrote) */
    const int32_t *dust_count; /* [n_total] packages sent from each cell (soc_oracle_emission_counts) */
    double dust_freq_hz;       /* frequency of this simulation, for B_nu(T) */
    double *dust_self;         /* f3, may be NULL: [n_total] += weight * energy a dust package deposits in the cell that
                                  emitted it before it first leaves that cell (the absorption-emission cycle inside a
                                  cell that the diagonal ALI operator solves explicitly) */
} soc_oracle_sources;

typedef struct {
    double emitted, escaped, absorbed;
    uint64_t cell_steps, scatterings, terminated;
} soc_oracle_result;

typedef struct {           /* per-package replay record */
    uint64_t hash;         /* FNV-style hash of the visited global cell ids */
    uint32_t steps, scatters;
    double e_escaped;
} soc_oracle_replay;

typedef struct {           /* one cell-step, global coordinates in root-cell units */
    int64_t pkg, gid;
    int32_t level, kind;   /* kind: 0 cross, 1 scatter, 2 terminated here, 3 cross and escape */
    double p0[3], p1[3];
    double ds, tau_sca;    /* path length and scattering optical depth of the step */
    double tau_drawn;      /* -ln u of the flight segment this step belongs to */
} soc_oracle_trace;

/* origin (lower corner, root units) of cell (level, c) by following the reverse links */
static void cell_origin(const soc_oracle_grid *G, int32_t level, int32_t c, double org[3])
{
    double h = ldexp(1.0, -(level - 1));
    double o[3] = { 0.0, 0.0, 0.0 };
    while (level > 1) {
        o[0] += h * (double)(c & 1);
        o[1] += h * (double)((c >> 1) & 1);
        o[2] += h * (double)((c >> 2) & 1);
        c = G->parent[level - 1][c >> 3];
        level -= 1;
        h *= 2.0;
    }
    int32_t ix = c % G->nx, iy = (c / G->nx) % G->ny, iz = c / (G->nx * G->ny);
    org[0] = o[0] + ix; org[1] = o[1] + iy; org[2] = o[2] + iz;
}

/* Descend to the leaf that holds the position ("down to the new leaf node").
 * f >= 0.5 goes to the upper child; 2f and 2f-1 are exact. */
static void descend(const soc_oracle_grid *G, soc_oracle_state *S)
{
    for (;;) {
        int32_t ch = G->child[G->level_off[S->level - 1] + S->cell];
        if (ch < 0) return;
        int32_t slot = 0;
        for (int j = 0; j < 3; ++j) {
            if (S->f[j] >= 0.5) { slot |= (1 << j); S->f[j] = 2.0 * S->f[j] - 1.0; }   /* exact, also in fp32 */
            else S->f[j] = 2.0 * S->f[j];
        }
        S->cell = ch + slot;
        S->level += 1;
    }
}

/* Move across the face of axis a in direction sg (+1/-1): sibling flip, else up to the
 * common parent, then down.  Returns 0 if the package left the root grid. */
static int move_across(const soc_oracle_grid *G, soc_oracle_state *S, int a, int sg)
{
    for (;;) {
        if (S->level == 1) {
            int32_t n[3] = { G->nx, G->ny, G->nz };
            int32_t i[3] = { S->cell % G->nx, (S->cell / G->nx) % G->ny, S->cell / (G->nx * G->ny) };
            i[a] += sg;
            if (i[a] < 0 || i[a] >= n[a]) return 0;
            S->cell = i[0] + G->nx * (i[1] + G->ny * i[2]);
            break;
        }
        int bit = (S->cell >> a) & 1;
        if ((sg > 0 && bit == 0) || (sg < 0 && bit == 1)) { S->cell ^= (1 << a); break; }
        for (int j = 0; j < 3; ++j) S->f[j] = keep((S->f[j] + (double)((S->cell >> j) & 1)) * 0.5, S->f32state);
        S->cell = G->parent[S->level - 1][S->cell >> 3];
        S->level -= 1;
    }
    S->f[a] = (sg > 0) ? 0.0 : 1.0;   /* entry face, in the neighbour's frame */
    descend(G, S);
    return 1;
}

/* ------------------------------------------------------------------ a2, a3: emission - */
/* Number of background packages and package energies (reading S3). */
static int64_t split_n_bg(const soc_oracle_sources *src, int64_t n_packages)
{
    if (src->n_bg >= 0) return src->n_bg;
    int has_bg = src->bg_intensity > 0.0, has_ps = src->n_point > 0;
    if (has_bg && has_ps) return n_packages / 2;
    return has_bg ? n_packages : 0;
}

/* Background: face chosen in proportion to its area, uniform point on
 * the face, cosine-law direction into the volume; E0 = pi I S / n_bg. */
void soc_oracle_emit_background(int32_t nx, int32_t ny, int32_t nz, const double u[5],
                                int32_t cell_ijk[3], double f[3], double d[3])
{
    double N[3] = { (double)nx, (double)ny, (double)nz };
    double area[3] = { N[1] * N[2], N[2] * N[0], N[0] * N[1] };   /* faces normal to x, y, z */
    double S = 2.0 * (area[0] + area[1] + area[2]);
    double x = u[0] * S, cum = 0.0;
    int face = 5;
    for (int k = 0; k < 6; ++k) { cum += area[k / 2]; if (x < cum) { face = k; break; } }
    int a = face / 2, a1 = (a + 1) % 3, a2 = (a + 2) % 3, high = face & 1;
    int32_t n_i[3] = { nx, ny, nz };
    double t1 = u[1] * N[a1], t2 = u[2] * N[a2];
    int32_t i1 = (int32_t)floor(t1); if (i1 > n_i[a1] - 1) i1 = n_i[a1] - 1;
    int32_t i2 = (int32_t)floor(t2); if (i2 > n_i[a2] - 1) i2 = n_i[a2] - 1;
    cell_ijk[a1] = i1; f[a1] = t1 - i1;
    cell_ijk[a2] = i2; f[a2] = t2 - i2;
    cell_ijk[a] = high ? n_i[a] - 1 : 0;
    f[a] = high ? 1.0 : 0.0;
    double mu = sqrt(u[3]), st = sqrt(1.0 - u[3]), phi = 2.0 * SOC_O_PI * u[4];
    d[a] = high ? -mu : mu;
    d[a1] = st * cos(phi);
    d[a2] = st * sin(phi);
}

/* Point source: fixed position, isotropic direction. */
void soc_oracle_emit_point(const double pos[3], const double u[2],
                           int32_t cell_ijk[3], double f[3], double d[3])
{
    for (int j = 0; j < 3; ++j) { cell_ijk[j] = (int32_t)floor(pos[j]); f[j] = pos[j] - cell_ijk[j]; }
    double mu = 2.0 * u[0] - 1.0, st = sqrt(fmax(0.0, 1.0 - mu * mu)), phi = 2.0 * SOC_O_PI * u[1];
    d[0] = st * cos(phi); d[1] = st * sin(phi); d[2] = mu;
}

/* ------------------------------------------------------------------ f1: dust re-emission
 * "If grains are assumed to be in an equilibrium with the radiation field, the emission is calculated by SOC itself"
 * (PAPER.md:67); the cells are then a third source of photon packages, needed when "dust is heated to such high
 * temperatures that its emission no longer freely escapes the model volume".
 * Luminosity of leaf c at frequency nu, in the energy unit of pi I S (lengths in root-cell edges):
 *     L_c = 4 pi kabs rho_c h_l^3 B_nu(T_c)            (kabs rho = absorption optical depth per unit length)
 * Package counts per cell are the host's policy (readings F1-F2 in DESIGN.md):
 *   mode 0, uniform:  "the same number of photon packages is sent per each cell", the total "a multiple of the number
 *                     of cells": m = ceil(n_request / n_emitting) packages from every cell with L_c > 0
 *   mode 1, weighted: "the number of emitted photon packages is weighted according to the emission", "the maximum
 *                     number of photon packages sent from any single cell was limited ... with a user-defined
 *                     parameter": n_c = min(cap, ceil(n_request L_c / sum L)) for L_c > 0
 * Each package of cell c carries L_c / n_c, so the emitted energy is exactly sum L_c whatever the counts. */
#define SOC_O_H  6.62607015e-27
#define SOC_O_KB 1.380649e-16
#define SOC_O_C  2.99792458e10

double soc_oracle_planck(double nu, double T)
{
    if (!(T > 0.0)) return 0.0;
    return 2.0 * SOC_O_H * nu * nu * nu / (SOC_O_C * SOC_O_C) / expm1(SOC_O_H * nu / (SOC_O_KB * T));
}

/* L_c for every cell (0 for parents, empty leaves and T <= 0).  lum: [n_total]. */
void soc_oracle_cell_luminosity(const soc_oracle_grid *G, double kabs, double freq_hz, const float *T, double *lum)
{
    for (int l = 1; l <= G->n_levels; ++l) {
        const double h = ldexp(1.0, -(l - 1)), vol = h * h * h;
        for (int64_t gid = G->level_off[l - 1]; gid < G->level_off[l]; ++gid) {
            const double rho = (double)G->rho[gid];
            lum[gid] = (G->child[gid] >= 0 || !(rho > 0.0)) ? 0.0
                     : 4.0 * SOC_O_PI * kabs * rho * vol * soc_oracle_planck(freq_hz, (double)T[gid]);
        }
    }
}

/* Package counts per cell; returns their sum (n_dust), or -1 on a bad argument. */
int64_t soc_oracle_emission_counts(const soc_oracle_grid *G, double kabs, double freq_hz, const float *T, int32_t mode,
                                   int64_t n_request, int32_t cap, int32_t *count)
{
    if (!G || !T || !count || n_request < 0 || (mode != 0 && mode != 1) || (mode == 1 && cap < 1)) return -1;
    double *lum = (double *)malloc(sizeof(double) * (size_t)G->n_total);
    soc_oracle_cell_luminosity(G, kabs, freq_hz, T, lum);
    double tot = 0.0;
    int64_t n_emit = 0, n_dust = 0;
    for (int64_t c = 0; c < G->n_total; ++c) { tot += lum[c]; n_emit += lum[c] > 0.0; }
    const int64_t m = n_emit > 0 ? (n_request + n_emit - 1) / n_emit : 0;
    for (int64_t c = 0; c < G->n_total; ++c) {
        int64_t n = 0;
        if (lum[c] > 0.0 && n_request > 0) {
            if (mode == 0) n = m;
            else { n = (int64_t)ceil((double)n_request * lum[c] / tot); if (n < 1) n = 1; if (n > cap) n = cap; }
        }
        count[c] = (int32_t)n;
        n_dust += n;
    }
    free(lum);
    return n_dust;
}

/* Stride that spreads consecutive dust package ids over the cells: the odd number nearest below n_dust / golden ratio
 * that is coprime to n_dust (so that q -> q * stride mod n_dust is a permutation of [0, n_dust)). */
int64_t soc_oracle_dust_stride(int64_t n_dust)
{
    if (n_dust <= 2) return 1;
    int64_t s = (int64_t)floor((double)n_dust * 0.6180339887498949) | 1;
    for (;;) {
        int64_t a = s, b = n_dust;
        while (b) { int64_t t = a % b; a = b; b = t; }
        if (a == 1) return s;
        s += 2;
    }
}

/* A dust package (readings F3): uniform point in the cell, isotropic direction -- "random locations and directions
 * within each cell".  u[0..2] -> position, u[3] -> cos(theta) = 2u - 1, u[4] -> azimuth. */
void soc_oracle_emit_cell(const double u[5], double f[3], double d[3])
{
    for (int j = 0; j < 3; ++j) f[j] = u[j];
    double mu = 2.0 * u[3] - 1.0, st = sqrt(fmax(0.0, 1.0 - mu * mu)), phi = 2.0 * SOC_O_PI * u[4];
    d[0] = st * cos(phi); d[1] = st * sin(phi); d[2] = mu;
}

/* ------------------------------------------------------------------ a4-a9: the walk - */
#define SOC_O_WMIN 1e-9   /* termination: weight below WMIN * E0, residual deposited (S7) */

/* Simulate package ids [pkg_begin, pkg_begin + pkg_count) of a run of n_packages at
 * frequency index ifreq.  absorbed[gid] += weight * (energy absorbed in the cell).
 * replay (may be NULL): pkg_count records.  trace (may be NULL): up to trace_cap steps,
 * *n_trace receives the number written.  Returns 0, or -1 on a bad argument. */
static int simulate(const soc_oracle_grid *G, double kabs, double ksca, double g, int32_t ifreq,
                    const soc_oracle_sources *src, int64_t n_packages, uint64_t seed, double weight,
                    int64_t pkg_begin, int64_t pkg_count, double *absorbed,
                    soc_oracle_result *res, soc_oracle_replay *replay,
                    soc_oracle_trace *trace, int64_t trace_cap, int64_t *n_trace, int32_t f32state)
{
    if (!G || !src || !absorbed || n_packages < 0 || pkg_begin < 0 || pkg_count < 0 ||
        pkg_begin + pkg_count > n_packages || !(kabs >= 0.0) || !(ksca >= 0.0) || !(fabs(g) < 1.0))
        return -1;
    /* ids [0, n_bg) background, [n_bg, n_packages - n_dust) point sources, the last n_dust ids dust re-emission */
    const int64_t n_dust = src->beam ? 0 : src->n_dust;
    if (n_dust < 0 || n_dust > n_packages) return -1;
    const int64_t n_const = n_packages - n_dust;
    const int64_t n_bg = src->beam ? 0 : split_n_bg(src, n_const);
    if (n_bg > n_const) return -1;
    int64_t *dust_first = NULL;      /* [n_total + 1] first dust index of every cell: prefix sums of dust_count */
    double *dust_lum = NULL;
    if (n_dust > 0) {
        if (!src->dust_T || !src->dust_count || !(src->dust_freq_hz > 0.0)) return -1;
        dust_first = (int64_t *)malloc(sizeof(int64_t) * (size_t)(G->n_total + 1));
        dust_lum = (double *)malloc(sizeof(double) * (size_t)G->n_total);
        soc_oracle_cell_luminosity(G, kabs, src->dust_freq_hz, src->dust_T, dust_lum);
        dust_first[0] = 0;
        for (int64_t c = 0; c < G->n_total; ++c) {
            if (src->dust_count[c] < 0 || (src->dust_count[c] > 0 && !(dust_lum[c] > 0.0))) { free(dust_first); free(dust_lum); return -1; }
            dust_first[c + 1] = dust_first[c] + src->dust_count[c];
        }
        if (dust_first[G->n_total] != n_dust || n_dust >= ((int64_t)1 << 32)) { free(dust_first); free(dust_lum); return -1; }
    }
    const int64_t dust_stride = soc_oracle_dust_stride(n_dust);
    if (!src->beam) {
        if (n_bg > 0 && !(src->bg_intensity > 0.0)) { free(dust_first); free(dust_lum); return -1; }
        if (n_const - n_bg > 0 && src->n_point <= 0) { free(dust_first); free(dust_lum); return -1; }
        for (int k = 0; k < src->n_point; ++k) {
            const double *p = src->ps_pos + 3 * k;
            if (!(p[0] > 0.0 && p[0] < G->nx && p[1] > 0.0 && p[1] < G->ny && p[2] > 0.0 && p[2] < G->nz)) { free(dust_first); free(dust_lum); return -1; }
        }
    }
    const double surf = 2.0 * ((double)G->ny * G->nz + (double)G->nz * G->nx + (double)G->nx * G->ny);
    soc_oracle_result R; memset(&R, 0, sizeof(R));
    int64_t nt = 0;

    for (int64_t p = pkg_begin; p < pkg_begin + pkg_count; ++p) {
        soc_oracle_state S;
        int32_t ijk[3];
        double E0, f0[3], d0[3];
        int64_t origin_gid = -1;                   /* dust package: the cell that emitted it */
        uint32_t w0[4], w1[4];
        soc_oracle_stream_block(seed, ifreq, p, 0u, w0);
        soc_oracle_stream_block(seed, ifreq, p, 1u, w1);
        if (src->beam) {
            E0 = 1.0;
            for (int j = 0; j < 3; ++j) {
                ijk[j] = (int32_t)floor(src->beam[j]);
                int32_t nj = (j == 0) ? G->nx : (j == 1) ? G->ny : G->nz;
                if (ijk[j] > nj - 1) ijk[j] = nj - 1;     /* a beam may start on the upper boundary */
                f0[j] = src->beam[j] - ijk[j];
                d0[j] = src->beam[3 + j];
            }
        } else if (p < n_bg) {
            double u[5] = { soc_oracle_uniform(w0[0]), soc_oracle_uniform(w0[1]), soc_oracle_uniform(w0[2]),
                            soc_oracle_uniform(w0[3]), soc_oracle_uniform(w1[0]) };
            soc_oracle_emit_background(G->nx, G->ny, G->nz, u, ijk, f0, d0);
            E0 = SOC_O_PI * src->bg_intensity * surf / (double)n_bg;
        } else if (p >= n_const) {
            /* f1: dust package q belongs to the cell c with dust_first[c] <= q < dust_first[c + 1] */
            /* (consecutive ids are spread over the cells -- q -> q * stride mod n_dust, stride coprime to n_dust --
             * as point-source ids are interleaved over the sources (S3): simultaneous packages of one cell are what
             * the paper blames for its GPU slow-down with emission weighting) */
            const int64_t q = (int64_t)(((uint64_t)(p - n_const) * (uint64_t)dust_stride) % (uint64_t)n_dust);
            int64_t lo = 0, hi = G->n_total;               /* invariant: dust_first[lo] <= q < dust_first[hi] */
            while (hi - lo > 1) { int64_t mid = (lo + hi) / 2; if (dust_first[mid] <= q) lo = mid; else hi = mid; }
            origin_gid = lo;
            double u[5] = { soc_oracle_uniform(w0[0]), soc_oracle_uniform(w0[1]), soc_oracle_uniform(w0[2]),
                            soc_oracle_uniform(w0[3]), soc_oracle_uniform(w1[0]) };
            soc_oracle_emit_cell(u, f0, d0);
            E0 = dust_lum[lo] / (double)src->dust_count[lo];
        } else {
            int64_t q = p - n_bg, n_ps = n_const - n_bg;
            int32_t k = (int32_t)(q % src->n_point);
            /* count_k = number of ids q in [0, n_ps) with q mod n_point == k */
            int64_t count_k = n_ps / src->n_point + ((n_ps % src->n_point) > k ? 1 : 0);
            double u[2] = { soc_oracle_uniform(w0[0]), soc_oracle_uniform(w0[1]) };
            soc_oracle_emit_point(src->ps_pos + 3 * k, u, ijk, f0, d0);
            E0 = src->ps_lum[k] / (double)count_k;
        }
        S.f32state = f32state;
        for (int j = 0; j < 3; ++j) { S.f[j] = keep(f0[j], f32state); S.d[j] = keep(d0[j], f32state); }
        if (origin_gid >= 0) {                         /* a dust package starts inside its (leaf) cell */
            int32_t l = 1;
            while (origin_gid >= G->level_off[l]) ++l;
            S.level = l;
            S.cell = (int32_t)(origin_gid - G->level_off[l - 1]);
        } else {
            S.level = 1;
            S.cell = ijk[0] + G->nx * (ijk[1] + G->ny * ijk[2]);
            descend(G, &S);
        }
        int in_origin = origin_gid >= 0;               /* f3: still inside the emitting cell, never left it */

        double E = E0;
        R.emitted += E0;
        uint32_t seg = 0, steps = 0, scat = 0;
        uint64_t hash = 0xcbf29ce484222325ull;
        double e_esc = 0.0;
        uint32_t ws[4];
        soc_oracle_stream_block(seed, ifreq, p, 2u + seg, ws);
        double tau_drawn = keep(-log(soc_oracle_uniform(ws[0])), f32state);   /* a4: free path, scattering depth */
        double tau_rem = tau_drawn;

        for (;;) {
            const int64_t gid = G->level_off[S.level - 1] + S.cell;
            const double rho = (double)G->rho[gid];
            const double h = ldexp(1.0, -(S.level - 1));
            /* a5/a6: distance (in cell edges) to the face of each axis */
            double t[3];
            for (int j = 0; j < 3; ++j) {
                const double fj = S.f[j], dj = S.d[j];
                if (dj > 0.0) t[j] = (1.0 - fj) / dj;
                else if (dj < 0.0) t[j] = (-fj) / dj;
                else t[j] = INFINITY;
                if (t[j] < 0.0) t[j] = 0.0;
            }
            int a = 0;                                    /* lowest axis wins a tie (S4) */
            if (t[1] < t[a]) a = 1;
            if (t[2] < t[a]) a = 2;
            const double tstar = t[a];
            const double ds = tstar * h;
            const double ks_rho = rho * ksca;
            const double dtau = ds * ks_rho;
            int scatter = 0;
            double ds_used = ds, t_used = tstar;
            if (ks_rho > 0.0 && dtau >= tau_rem) {
                scatter = 1;
                ds_used = tau_rem / ks_rho;
                t_used = ds_used / h;
            }
            /* a7: path-length estimator, continuous absorption */
            const double dep = E * (-expm1(-ds_used * rho * kabs));
            absorbed[gid] += weight * dep;
            if (in_origin && src->dust_self) src->dust_self[gid] += weight * dep;
            R.absorbed += dep;
            E -= dep;
            steps += 1;
            hash = (hash ^ (uint64_t)gid) * 0x100000001b3ull;

            soc_oracle_trace *T = NULL;
            if (trace && nt < trace_cap) {
                T = &trace[nt++];
                double org[3];
                cell_origin(G, S.level, S.cell, org);
                T->pkg = p; T->gid = gid; T->level = S.level; T->kind = scatter ? 1 : 0;
                for (int j = 0; j < 3; ++j) T->p0[j] = org[j] + h * S.f[j];
                T->ds = ds_used; T->tau_sca = ds_used * ks_rho; T->tau_drawn = tau_drawn;
            }
            /* a9: termination */
            if (E < SOC_O_WMIN * E0) {
                absorbed[gid] += weight * E;
                if (in_origin && src->dust_self) src->dust_self[gid] += weight * E;
                R.absorbed += E;
                E = 0.0;
                R.terminated += 1;
                if (T) { T->kind = 2; for (int j = 0; j < 3; ++j) T->p1[j] = T->p0[j] + ds_used * S.d[j]; }
                break;
            }
            for (int j = 0; j < 3; ++j) {
                double fn = S.f[j] + t_used * S.d[j];
                if (fn < 0.0) fn = 0.0;
                if (fn > 1.0) fn = 1.0;
                S.f[j] = keep(fn, f32state);
            }
            if (T) {
                double org[3];
                cell_origin(G, S.level, S.cell, org);
                for (int j = 0; j < 3; ++j) T->p1[j] = org[j] + h * S.f[j];
            }
            if (scatter) {
                /* a8 */
                double cost = soc_oracle_hg_cos(g, soc_oracle_uniform(ws[1]));
                double phi = 2.0 * SOC_O_PI * soc_oracle_uniform(ws[2]);
                double nd[3];
                soc_oracle_rotate(S.d, cost, phi, nd);
                for (int j = 0; j < 3; ++j) S.d[j] = keep(nd[j], f32state);
                seg += 1; scat += 1;
                soc_oracle_stream_block(seed, ifreq, p, 2u + seg, ws);
                tau_drawn = keep(-log(soc_oracle_uniform(ws[0])), f32state);
                tau_rem = tau_drawn;
            } else {
                tau_rem = keep(tau_rem - dtau, f32state);
                in_origin = 0;                           /* the package leaves the cell it is in */
                if (!move_across(G, &S, a, S.d[a] > 0.0 ? 1 : -1)) {
                    e_esc = E;                           /* a9: escape */
                    R.escaped += E;
                    if (T) T->kind = 3;
                    break;
                }
            }
        }
        R.cell_steps += steps;
        R.scatterings += scat;
        if (replay) {
            soc_oracle_replay *rp = &replay[p - pkg_begin];
            rp->hash = hash; rp->steps = steps; rp->scatters = scat; rp->e_escaped = e_esc;
        }
    }
    free(dust_first); free(dust_lum);
    if (res) *res = R;
    if (n_trace) *n_trace = nt;
    return 0;
}

/* THE oracle: fp64 throughout (north_star). */
int soc_oracle_simulate(const soc_oracle_grid *G, double kabs, double ksca, double g, int32_t ifreq,
                        const soc_oracle_sources *src, int64_t n_packages, uint64_t seed, double weight,
                        int64_t pkg_begin, int64_t pkg_count, double *absorbed,
                        soc_oracle_result *res, soc_oracle_replay *replay,
                        soc_oracle_trace *trace, int64_t trace_cap, int64_t *n_trace)
{
    return simulate(G, kabs, ksca, g, ifreq, src, n_packages, seed, weight, pkg_begin, pkg_count, absorbed, res,
                    replay, trace, trace_cap, n_trace, 0);
}

/* The same walk with the package state snapped to fp32 at every store (header, "Precision"): used by the
 * replay-parity tests only, pinned to soc_oracle_simulate by tests/test_oracle_pins.py. */
int soc_oracle_simulate_f32state(const soc_oracle_grid *G, double kabs, double ksca, double g, int32_t ifreq,
                                 const soc_oracle_sources *src, int64_t n_packages, uint64_t seed, double weight,
                                 int64_t pkg_begin, int64_t pkg_count, double *absorbed,
                                 soc_oracle_result *res, soc_oracle_replay *replay,
                                 soc_oracle_trace *trace, int64_t trace_cap, int64_t *n_trace)
{
    return simulate(G, kabs, ksca, g, ifreq, src, n_packages, seed, weight, pkg_begin, pkg_count, absorbed, res,
                    replay, trace, trace_cap, n_trace, 1);
}

/* ------------------------------------------------------------------ a10 -------------
 * Trapezoid weights in nu on the given grid (PAPER.md:67 only says the integral over
 * frequency is gathered during the simulation; quadrature = reading S9). */
void soc_oracle_trapezoid_weights(const double *freq, int32_t n, double *w)
{
    if (n == 1) { w[0] = 1.0; return; }
    for (int i = 0; i < n; ++i) {
        double lo = freq[i > 0 ? i - 1 : 0], hi = freq[i < n - 1 ? i + 1 : n - 1];
        w[i] = 0.5 * fabs(hi - lo);
    }
}

/* ------------------------------------------------------------------ a11 -------------
 * Energy balance by table lookup (table form = reading S10).
 * E_c = scale * Aint_c / (rho_c h_l^3); table T_k on E_k = E_min (E_max/E_min)^(k/(n-1));
 * linear interpolation in the table index; E_c <= E_min (also unhit cells) -> T_0;
 * E_c >= E_max -> T_{n-1}; rho = 0 leaves and parent cells -> 0. */
void soc_oracle_update_temperatures(const soc_oracle_grid *G, const double *absorbed, double scale,
                                    const float *table_T, int32_t n_table, double E_min, double E_max,
                                    float *T_out)
{
    const double lmin = log(E_min), lmax = log(E_max);
    for (int l = 1; l <= G->n_levels; ++l) {
        const double h = ldexp(1.0, -(l - 1)), vol = h * h * h;
        for (int64_t gid = G->level_off[l - 1]; gid < G->level_off[l]; ++gid) {
            const double rho = (double)G->rho[gid];
            if (G->child[gid] >= 0 || !(rho > 0.0)) { T_out[gid] = 0.0f; continue; }
            const double Ec = scale * absorbed[gid] / (rho * vol);
            double T;
            if (!(Ec > E_min)) T = (double)table_T[0];
            else if (Ec >= E_max) T = (double)table_T[n_table - 1];
            else {
                double x = (log(Ec) - lmin) / (lmax - lmin) * (double)(n_table - 1);
                int32_t i = (int32_t)floor(x);
                if (i > n_table - 2) i = n_table - 2;
                if (i < 0) i = 0;
                T = (double)table_T[i] + (x - (double)i) * ((double)table_T[i + 1] - (double)table_T[i]);
            }
            T_out[gid] = (float)T;
        }
    }
}

/* ------------------------------------------------------------------ f3: ALI ---------
 * Accelerated lambda iteration "with a diagonal operator that solves explicitly for the cycle of photons that are
 * absorbed within the emitting cell", at the cost of "one additional floating point number per cell, which is needed
 * to keep track of the photon escape probabilities for each cell".  Reading F6:
 *   self_c    = frequency-integrated energy that the cell's own packages deposited in it before first leaving it
 *   emitted_c = frequency-integrated energy the cell emitted in that simulation (sum_f w_f L_c,f at the OLD temperature)
 *   beta_c    = self_c / emitted_c                 (1 - beta_c = the cell's photon escape probability)
 * Energy balance with the in-cell cycle taken out:  Lambda(T_new) rho V (1 - beta_c) = absorbed_c - self_c, i.e. the
 * table is entered with  E_c = scale (absorbed_c - self_c) / (rho_c h^3 (1 - beta_c)).  beta_c = 0 gives a11 back. */
void soc_oracle_update_temperatures_ali(const soc_oracle_grid *G, const double *absorbed, const double *self_abs,
                                        const double *emitted, double scale, const float *table_T, int32_t n_table,
                                        double E_min, double E_max, float *T_out)
{
    double *eff = (double *)malloc(sizeof(double) * (size_t)G->n_total);
    for (int64_t c = 0; c < G->n_total; ++c) {
        double beta = (emitted[c] > 0.0) ? self_abs[c] / emitted[c] : 0.0;
        if (beta > 0.999) beta = 0.999;            /* a cell that keeps everything: bounded acceleration */
        if (beta < 0.0) beta = 0.0;
        eff[c] = (absorbed[c] - self_abs[c]) / (1.0 - beta);
        if (eff[c] < 0.0) eff[c] = 0.0;
    }
    soc_oracle_update_temperatures(G, eff, scale, table_T, n_table, E_min, E_max, T_out);
    free(eff);
}

/* ------------------------------------------------------------------ f2: maps --------
 * "As the final step, the host calls a mapping kernel to make surface brightness maps for the desired frequencies and
 * directions" (K3 of PAPER.md:55; 1310 x 1310 pixels of the size of the smallest cells).
 * The paper gives no formula; reading M1: thermal dust emission integrated along parallel lines of sight
 * with extinction by absorption + scattering, no background behind the cloud, no scattered light (the paper makes
 * those "with separate runs"):
 *     I = sum over the cells k crossed, front to back, of  exp(-tau_k) S_k (1 - exp(-dtau_k)),
 *     dtau_k = (kabs + ksca) rho_k ds_k,  S_k = kabs / (kabs + ksca) B_nu(T_k),  tau_k = sum of dtau in front of k.
 * Geometry (reading M2): orthographic.  Pixel (i, j), i < npx fastest, looks along the unit vector dir from the point
 *     o = centre + ((i + 1/2) - npx/2) pixel ex + ((j + 1/2) - npy/2) pixel ey          (ex, ey, dir orthonormal)
 * The line enters the root grid where the slab test says; the cells are walked exactly as the packages walk them (a5/a6). */
void soc_oracle_make_map(const soc_oracle_grid *G, double kabs, double ksca, double freq_hz, const float *T,
                         const double ex[3], const double ey[3], const double dir[3], const double centre[3],
                         int32_t npx, int32_t npy, double pixel, double *map)
{
    const double N[3] = { (double)G->nx, (double)G->ny, (double)G->nz };
    const double kext = kabs + ksca;
    for (int32_t j = 0; j < npy; ++j) for (int32_t i = 0; i < npx; ++i) {
        const double a = ((double)i + 0.5 - 0.5 * (double)npx) * pixel, b = ((double)j + 0.5 - 0.5 * (double)npy) * pixel;
        double o[3], t_in = -INFINITY, t_out = INFINITY;
        for (int k = 0; k < 3; ++k) o[k] = centre[k] + a * ex[k] + b * ey[k];
        for (int k = 0; k < 3; ++k) {                       /* slab test against [0, N_k] */
            if (dir[k] != 0.0) {
                double t0 = (0.0 - o[k]) / dir[k], t1 = (N[k] - o[k]) / dir[k];
                if (t0 > t1) { double t = t0; t0 = t1; t1 = t; }
                if (t0 > t_in) t_in = t0;
                if (t1 < t_out) t_out = t1;
            } else if (o[k] < 0.0 || o[k] > N[k]) { t_in = INFINITY; }
        }
        double I = 0.0, tau = 0.0;
        if (t_in < t_out) {
            soc_oracle_state S;
            S.f32state = 0;
            int32_t ijk[3];
            for (int k = 0; k < 3; ++k) {
                double x = o[k] + t_in * dir[k];
                int32_t c = (int32_t)floor(x);
                const int32_t nk = (k == 0) ? G->nx : (k == 1) ? G->ny : G->nz;
                if (c < 0) c = 0;
                if (c > nk - 1) c = nk - 1;
                double f = x - (double)c;
                if (f < 0.0) f = 0.0;
                if (f > 1.0) f = 1.0;
                ijk[k] = c; S.f[k] = f; S.d[k] = dir[k];
            }
            S.level = 1;
            S.cell = ijk[0] + G->nx * (ijk[1] + G->ny * ijk[2]);
            descend(G, &S);
            for (;;) {
                const int64_t gid = G->level_off[S.level - 1] + S.cell;
                const double h = ldexp(1.0, -(S.level - 1));
                double t[3];
                for (int k = 0; k < 3; ++k) {
                    if (S.d[k] > 0.0) t[k] = (1.0 - S.f[k]) / S.d[k];
                    else if (S.d[k] < 0.0) t[k] = (-S.f[k]) / S.d[k];
                    else t[k] = INFINITY;
                    if (t[k] < 0.0) t[k] = 0.0;
                }
                int ax = 0;
                if (t[1] < t[ax]) ax = 1;
                if (t[2] < t[ax]) ax = 2;
                const double ds = t[ax] * h, rho = (double)G->rho[gid];
                const double dtau = kext * rho * ds;
                if (dtau > 0.0 && (double)T[gid] > 0.0)
                    I += exp(-tau) * (kabs / kext) * soc_oracle_planck(freq_hz, (double)T[gid]) * (-expm1(-dtau));
                tau += dtau;
                for (int k = 0; k < 3; ++k) {
                    double fn = S.f[k] + t[ax] * S.d[k];
                    if (fn < 0.0) fn = 0.0;
                    if (fn > 1.0) fn = 1.0;
                    S.f[k] = fn;
                }
                if (!move_across(G, &S, ax, S.d[ax] > 0.0 ? 1 : -1)) break;
            }
        }
        map[(int64_t)j * npx + i] = I;
    }
}

int64_t soc_oracle_sizeof_replay(void) { return (int64_t)sizeof(soc_oracle_replay); }
int64_t soc_oracle_sizeof_trace(void) { return (int64_t)sizeof(soc_oracle_trace); }
int64_t soc_oracle_grid_n_total(const soc_oracle_grid *G) { return G->n_total; }
const int32_t *soc_oracle_grid_parent(const soc_oracle_grid *G, int32_t level) { return G->parent[level - 1]; }
