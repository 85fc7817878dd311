/*
 * tpcgen.c -- seeded synthetic TPC workload generator (inputs only).
 *
 * This module serves BOTH the CPU oracle (oracle/) and the CUDA library with identical input
 * bytes.  It holds none of the track-finding arithmetic: it draws particles, intersects closed-form
 * helices with the pad rows of each sector (double precision), smears, drops, adds noise, shuffles
 * and stores fp32 (pad-y, time, charge) per (sector,row) plus the truth labels.
 *
 * Workload shapes follow BASELINE.json:configs[0..4] under the readings A20-A25 of SURVEY.md
 * section 8(c)/(d) (restated in DESIGN.md section 5): the paper measured on ALICE Pb-Pb / pp data and
 * Monte-Carlo, which are not available; these inputs stand in for them.
 *
 * Random numbers: counter-seeded splitmix64 streams (one per particle / per noise block), so the
 * output does not depend on the number of OpenMP threads.
 *
 * Build: gcc -O2 -fopenmp -shared -fPIC gen/tpcgen.c -o gen/libtpcgen.so -lm
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define TPCGEN_PI 3.14159265358979323846
#define TPCGEN_N_PHI_SECTORS 18
#define TPCGEN_N_SECTORS 36

typedef struct {
  uint64_t seed;
  int32_t n_rows;           /* 152 */
  int32_t single_sector;    /* 1: only sector 0 is read out, both z sides folded into it (config 1) */
  double x_first, x_last;   /* 85, 246 cm: radii of first/last pad row, rows evenly spaced */
  double bz;                /* Tesla */
  double vdrift;            /* cm/us */
  double z_max;             /* drift length, cm */
  double t_frame;           /* us; 0 = triggered single event; >0 = continuous time frame */
  double sigma_y, sigma_z;  /* Gaussian smearing, cm */
  double dropout;           /* Bernoulli probability that a crossing leaves no cluster */
  /* collisions */
  double rate_per_us;       /* t_frame>0: Poisson arrival rate (0.05 = 50 kHz) */
  int32_t mult_fixed;       /* >0: fixed number of primaries per collision */
  double mult_mean;         /* else ceil(Exp(mean)) ... */
  int32_t mult_cap;         /* ... capped here */
  double pt_lo, pt_hi;      /* primaries: log-uniform pT in GeV/c */
  double eta_max;           /* uniform in [-eta_max, eta_max] */
  double phi_lo, phi_hi;    /* primaries: uniform global azimuth range, rad */
  double sec_frac;          /* secondaries per primary */
  double sec_rmax;          /* secondary vertex radius uniform in [0, sec_rmax] */
  /* loopers (config 4) */
  int32_t n_loopers;        /* extra low-pT tracks per collision */
  double loop_pt_lo, loop_pt_hi; /* uniform pT */
  int32_t loop_turns;       /* max turns followed for loopers */
  /* noise */
  int32_t noise_per_sector; /* fixed count per active sector */
  double noise_frac;        /* plus this fraction of the track clusters, uniform over all units */
} tpcgen_params;

typedef struct {
  int32_t n_sectors, n_rows;
  int64_t n_clusters;
  int32_t n_particles, n_collisions;
  float* row_x;        /* [n_rows] */
  int64_t* unit_off;   /* [n_sectors*n_rows+1], unit = sector*n_rows+row */
  float* y;            /* [n] pad-y, cm (sector-local) */
  float* t;            /* [n] time, us */
  float* q;            /* [n] charge (never read by the tracker) */
  int32_t* label;      /* [n] particle id, -1 = noise */
  uint8_t* leg0;       /* [n] 1 = on the first outgoing leg of its particle */
  /* particle truth, [n_particles] each */
  int32_t* p_collision;
  int32_t* p_kind;     /* 0 primary, 1 secondary, 2 looper */
  int32_t* p_charge;
  double* p_pt; double* p_tanl; double* p_phi; double* p_t0;
  double* p_vx; double* p_vy; double* p_vz;
  int32_t* p_n_clusters;    /* all clusters left by the particle */
  int32_t* p_best_sector;   /* sector with most leg0 clusters, -1 if none */
  int32_t* p_best_count;    /* leg0 clusters in that sector */
  double* coll_t0;          /* [n_collisions] */
  int32_t* coll_mult;       /* [n_collisions] primaries */
} tpcgen_out;

/* ---------------- random numbers ---------------- */
static inline uint64_t mix64(uint64_t z) {
  z += 0x9E3779B97F4A7C15ULL;
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
  return z ^ (z >> 31);
}
typedef struct { uint64_t s; } rng_t;
static inline rng_t rng_make(uint64_t seed, uint64_t a, uint64_t b) {
  rng_t r; r.s = mix64(mix64(mix64(seed) ^ (a * 0xD1342543DE82EF95ULL)) ^ (b * 0xA24BAED4963EE407ULL)); return r;
}
static inline uint64_t rng_u64(rng_t* r) { r->s += 0x9E3779B97F4A7C15ULL; uint64_t z = r->s;
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL; z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL; return z ^ (z >> 31); }
static inline double rng_uni(rng_t* r) { return ((double)(rng_u64(r) >> 11) + 0.5) * (1.0 / 9007199254740992.0); }
static inline double rng_gauss(rng_t* r) { double u = rng_uni(r), v = rng_uni(r);
  return sqrt(-2.0 * log(u)) * cos(2.0 * TPCGEN_PI * v); }
static inline double rng_exp(rng_t* r) { return -log(rng_uni(r)); }

/* ---------------- growable cluster buffer ---------------- */
typedef struct { int32_t unit; float y, t, q; int32_t label; uint8_t leg0; } cl_t;
typedef struct { cl_t* a; int64_t n, cap; } clbuf_t;
static int clbuf_push(clbuf_t* b, cl_t c) {
  if (b->n == b->cap) { int64_t nc = b->cap ? b->cap * 2 : 4096; cl_t* na = (cl_t*)realloc(b->a, (size_t)nc * sizeof(cl_t));
    if (!na) return -1; b->a = na; b->cap = nc; }
  b->a[b->n++] = c; return 0;
}

typedef struct { int32_t collision, kind, charge; double pt, tanl, phi, t0, vx, vy, vz; } part_t;

static double wrap_pi(double a) { while (a > TPCGEN_PI) a -= 2 * TPCGEN_PI; while (a <= -TPCGEN_PI) a += 2 * TPCGEN_PI; return a; }

/* Clusters of one particle: every crossing of its helix with x_local = x_r inside each sector's wedge. */
static int gen_particle(const tpcgen_params* P, const double* row_x, const part_t* pa, int32_t pid, int turns,
                        clbuf_t* out, int32_t* leg0_count /* [36] */, int32_t* n_made) {
  const double cB = -0.00299792458 * P->bz;
  const double k = cB * (double)pa->charge / pa->pt;
  const double tan_half = tan(TPCGEN_PI / TPCGEN_N_PHI_SECTORS);
  const double dphi = 2 * TPCGEN_PI / TPCGEN_N_PHI_SECTORS;
  rng_t rc = rng_make(P->seed, 0x1000000ULL + (uint64_t)pid, 77);
  for (int ps = 0; ps < TPCGEN_N_PHI_SECTORS; ps++) {
    if (P->single_sector && ps != 0) continue;
    const double alpha = (ps + 0.5) * dphi;
    const double ca = cos(alpha), sa = sin(alpha);
    const double x0 = pa->vx * ca + pa->vy * sa, y0 = -pa->vx * sa + pa->vy * ca;
    const double phl = wrap_pi(pa->phi - alpha);
    const double s0 = sin(phl), c0 = cos(phl);
    if (k != 0.0) { /* can the circle reach the first row in this frame at all? */
      double xa = x0 + (-1.0 - s0) / k, xb = x0 + (1.0 - s0) / k;
      double xmax = xa > xb ? xa : xb;
      if (xmax < row_x[0]) continue;
    } else if (c0 <= 0) continue;
    for (int m = 0; m < turns; m++) {
      for (int b = 0; b < 2; b++) {
        for (int r = 0; r < P->n_rows; r++) {
          double xr = row_x[r], yy, l; int first_leg = 0;
          if (k == 0.0) {
            if (b || m) continue;
            l = (xr - x0) / c0; if (!(l > 0)) continue;
            yy = y0 + l * s0; first_leg = 1;
          } else {
            double s1 = s0 + k * (xr - x0);
            if (!(fabs(s1) < 1.0)) continue;
            double c1 = sqrt(1.0 - s1 * s1); if (b) c1 = -c1;
            yy = y0 - (c1 - c0) / k;
            if (fabs(yy) > xr * tan_half) continue;
            double a = asin(s1), psi = b ? (TPCGEN_PI - a) : a;
            double d = psi - phl;              /* turning angle, to be brought to the sign of k */
            if (k > 0) { while (d <= 0) d += 2 * TPCGEN_PI; while (d > 2 * TPCGEN_PI) d -= 2 * TPCGEN_PI; d += 2 * TPCGEN_PI * m; }
            else       { while (d >= 0) d -= 2 * TPCGEN_PI; while (d < -2 * TPCGEN_PI) d += 2 * TPCGEN_PI; d -= 2 * TPCGEN_PI * m; }
            l = d / k;
            first_leg = (b == 0 && m == 0 && c0 > 0 && fabs(d) < TPCGEN_PI);
          }
          if (fabs(yy) > xr * tan_half) continue;
          double zz = pa->vz + pa->tanl * l;
          if (fabs(zz) > P->z_max) continue;
          /* a crossing exists: draw in fixed order so the stream is reproducible */
          double u_drop = rng_uni(&rc), gy = rng_gauss(&rc), gz = rng_gauss(&rc), uq = rng_uni(&rc);
          if (u_drop < P->dropout) continue;
          double ym = yy + P->sigma_y * gy;
          double zabs = fabs(zz) + P->sigma_z * gz;      /* drift-frame z of the sector */
          double tt = pa->t0 + (P->z_max - zabs) / P->vdrift;
          if (P->t_frame > 0 && !(tt >= 0 && tt < P->t_frame)) continue;   /* outside the read-out frame */
          int side = (zz >= 0) ? 0 : 1;
          int sector = P->single_sector ? 0 : side * TPCGEN_N_PHI_SECTORS + ps;
          cl_t c; c.unit = sector * P->n_rows + r; c.y = (float)ym; c.t = (float)tt; c.q = (float)(10.0 + 90.0 * uq);
          c.label = pid; c.leg0 = (uint8_t)first_leg;
          if (clbuf_push(out, c)) return -1;
          if (first_leg) leg0_count[sector]++;
          (*n_made)++;
        }
      }
    }
  }
  return 0;
}

static int cmp_u64pair(const void* a, const void* b) {
  const uint64_t* x = (const uint64_t*)a; const uint64_t* y = (const uint64_t*)b;
  if (x[0] < y[0]) return -1; if (x[0] > y[0]) return 1;
  if (x[1] < y[1]) return -1; if (x[1] > y[1]) return 1; return 0;
}

void tpcgen_free(tpcgen_out* o) {
  if (!o) return;
  free(o->row_x); free(o->unit_off); free(o->y); free(o->t); free(o->q); free(o->label); free(o->leg0);
  free(o->p_collision); free(o->p_kind); free(o->p_charge); free(o->p_pt); free(o->p_tanl); free(o->p_phi); free(o->p_t0);
  free(o->p_vx); free(o->p_vy); free(o->p_vz); free(o->p_n_clusters); free(o->p_best_sector); free(o->p_best_count);
  free(o->coll_t0); free(o->coll_mult);
  memset(o, 0, sizeof(*o));
}

int tpcgen_generate(const tpcgen_params* P, tpcgen_out* o) {
  memset(o, 0, sizeof(*o));
  if (!P || P->n_rows < 3 || !(P->vdrift > 0) || !(P->z_max > 0) || !(P->pt_lo > 0) || !(P->pt_hi >= P->pt_lo)) return -1;
  const int R = P->n_rows, NS = TPCGEN_N_SECTORS, U = NS * R;
  o->n_sectors = NS; o->n_rows = R;
  double* row_x = (double*)malloc(sizeof(double) * R);
  o->row_x = (float*)malloc(sizeof(float) * R);
  for (int r = 0; r < R; r++) { row_x[r] = P->x_first + r * (P->x_last - P->x_first) / (R - 1); o->row_x[r] = (float)row_x[r]; }

  /* ---- collisions ---- */
  rng_t rg = rng_make(P->seed, 1, 1);
  int ncoll = 0, capc = 16; double* ct0 = (double*)malloc(sizeof(double) * capc); int32_t* cm = (int32_t*)malloc(sizeof(int32_t) * capc);
  if (P->t_frame > 0 && P->rate_per_us > 0) {
    double tt = 0;
    for (;;) { tt += rng_exp(&rg) / P->rate_per_us; if (tt >= P->t_frame) break;
      if (ncoll == capc) { capc *= 2; ct0 = (double*)realloc(ct0, sizeof(double) * capc); cm = (int32_t*)realloc(cm, sizeof(int32_t) * capc); }
      ct0[ncoll] = tt; cm[ncoll] = 0; ncoll++; }
  } else { ct0[0] = 0; cm[0] = 0; ncoll = 1; }
  int64_t npart = 0;
  for (int c = 0; c < ncoll; c++) {
    int m = P->mult_fixed;
    if (m <= 0) { double e = ceil(P->mult_mean * rng_exp(&rg)); if (e > P->mult_cap) e = P->mult_cap; if (e < 1) e = 1; m = (int)e; }
    cm[c] = m; npart += m + (int64_t)floor(m * P->sec_frac + 0.5) + P->n_loopers;
  }
  o->n_collisions = ncoll; o->coll_t0 = ct0; o->coll_mult = cm; o->n_particles = (int32_t)npart;

  /* ---- particles ---- */
  part_t* parts = (part_t*)malloc(sizeof(part_t) * (size_t)(npart > 0 ? npart : 1));
  { int64_t id = 0;
    for (int c = 0; c < ncoll; c++) {
      int nprim = cm[c], nsec = (int)floor(nprim * P->sec_frac + 0.5), nloop = P->n_loopers;
      for (int i = 0; i < nprim + nsec + nloop; i++, id++) {
        rng_t r = rng_make(P->seed, 0x2000000ULL + (uint64_t)id, 5);
        part_t* p = &parts[id]; p->collision = c; p->t0 = ct0[c];
        p->kind = i < nprim ? 0 : (i < nprim + nsec ? 1 : 2);
        if (p->kind == 2) p->pt = P->loop_pt_lo + (P->loop_pt_hi - P->loop_pt_lo) * rng_uni(&r);
        else p->pt = P->pt_lo * pow(P->pt_hi / P->pt_lo, rng_uni(&r));
        p->charge = rng_uni(&r) < 0.5 ? -1 : 1;
        p->tanl = sinh(P->eta_max * (2 * rng_uni(&r) - 1));
        p->phi = P->phi_lo + (P->phi_hi - P->phi_lo) * rng_uni(&r);
        p->vx = p->vy = p->vz = 0;
        if (p->kind == 1) { double rv = P->sec_rmax * rng_uni(&r), pv = 2 * TPCGEN_PI * rng_uni(&r), ev = P->eta_max * (2 * rng_uni(&r) - 1);
          p->vx = rv * cos(pv); p->vy = rv * sin(pv); p->vz = rv * sinh(ev); p->phi = 2 * TPCGEN_PI * rng_uni(&r); }
      }
    }
  }
  o->p_collision = (int32_t*)malloc(sizeof(int32_t) * (npart + 1)); o->p_kind = (int32_t*)malloc(sizeof(int32_t) * (npart + 1));
  o->p_charge = (int32_t*)malloc(sizeof(int32_t) * (npart + 1)); o->p_pt = (double*)malloc(sizeof(double) * (npart + 1));
  o->p_tanl = (double*)malloc(sizeof(double) * (npart + 1)); o->p_phi = (double*)malloc(sizeof(double) * (npart + 1));
  o->p_t0 = (double*)malloc(sizeof(double) * (npart + 1)); o->p_vx = (double*)malloc(sizeof(double) * (npart + 1));
  o->p_vy = (double*)malloc(sizeof(double) * (npart + 1)); o->p_vz = (double*)malloc(sizeof(double) * (npart + 1));
  o->p_n_clusters = (int32_t*)calloc(npart + 1, sizeof(int32_t)); o->p_best_sector = (int32_t*)malloc(sizeof(int32_t) * (npart + 1));
  o->p_best_count = (int32_t*)calloc(npart + 1, sizeof(int32_t));
  for (int64_t i = 0; i < npart; i++) { part_t* p = &parts[i];
    o->p_collision[i] = p->collision; o->p_kind[i] = p->kind; o->p_charge[i] = p->charge; o->p_pt[i] = p->pt; o->p_tanl[i] = p->tanl;
    o->p_phi[i] = p->phi; o->p_t0[i] = p->t0; o->p_vx[i] = p->vx; o->p_vy[i] = p->vy; o->p_vz[i] = p->vz; o->p_best_sector[i] = -1; }

  /* ---- track clusters: static contiguous chunks of particles per thread, concatenated in order ---- */
  int nthreads = 1;
#ifdef _OPENMP
  nthreads = omp_get_max_threads();
#endif
  if (nthreads > 64) nthreads = 64;
  clbuf_t* bufs = (clbuf_t*)calloc(nthreads, sizeof(clbuf_t));
  int fail = 0;
#pragma omp parallel num_threads(nthreads)
  {
    int tid = 0;
#ifdef _OPENMP
    tid = omp_get_thread_num();
#endif
    int64_t lo = npart * tid / nthreads, hi = npart * (tid + 1) / nthreads;
    for (int64_t i = lo; i < hi; i++) {
      int32_t cnt[TPCGEN_N_SECTORS]; memset(cnt, 0, sizeof(cnt)); int32_t made = 0;
      int turns = parts[i].kind == 2 ? P->loop_turns : 1;
      if (gen_particle(P, row_x, &parts[i], (int32_t)i, turns, &bufs[tid], cnt, &made)) { fail = 1; break; }
      int best = -1, bc = 0; for (int s = 0; s < NS; s++) if (cnt[s] > bc) { bc = cnt[s]; best = s; }
      o->p_n_clusters[i] = made; o->p_best_sector[i] = best; o->p_best_count[i] = bc;
    }
  }
  if (fail) { for (int t = 0; t < nthreads; t++) free(bufs[t].a); free(bufs); free(parts); free(row_x); tpcgen_free(o); return -2; }
  int64_t ntrk = 0; for (int t = 0; t < nthreads; t++) ntrk += bufs[t].n;

  /* ---- noise ---- */
  const int n_active = P->single_sector ? 1 : NS;
  int64_t nnoise = (int64_t)P->noise_per_sector * n_active + (int64_t)floor(P->noise_frac * (double)ntrk + 0.5);
  int64_t N = ntrk + nnoise;
  cl_t* all = (cl_t*)malloc(sizeof(cl_t) * (size_t)(N > 0 ? N : 1));
  { int64_t pos = 0; for (int t = 0; t < nthreads; t++) { if (bufs[t].n) memcpy(all + pos, bufs[t].a, sizeof(cl_t) * (size_t)bufs[t].n); pos += bufs[t].n; free(bufs[t].a); } }
  free(bufs);
  const double tan_half = tan(TPCGEN_PI / TPCGEN_N_PHI_SECTORS);
  const double t_drift = P->z_max / P->vdrift;
#pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < nnoise; i++) {
    rng_t r = rng_make(P->seed, 0x3000000ULL + (uint64_t)i, 9);
    int sector = (int)(rng_uni(&r) * n_active); if (sector >= n_active) sector = n_active - 1;
    int row = (int)(rng_uni(&r) * R); if (row >= R) row = R - 1;
    double yy = (2 * rng_uni(&r) - 1) * row_x[row] * tan_half;
    double tt = P->t_frame > 0 ? rng_uni(&r) * P->t_frame : rng_uni(&r) * t_drift;
    cl_t c; c.unit = sector * R + row; c.y = (float)yy; c.t = (float)tt; c.q = (float)(10.0 + 90.0 * rng_uni(&r)); c.label = -1; c.leg0 = 0;
    all[ntrk + i] = c;
  }

  /* ---- bucket by unit (stable), then shuffle inside each unit by a hash of the pre-shuffle index ---- */
  o->unit_off = (int64_t*)calloc((size_t)U + 1, sizeof(int64_t));
  for (int64_t i = 0; i < N; i++) o->unit_off[all[i].unit + 1]++;
  for (int u = 0; u < U; u++) o->unit_off[u + 1] += o->unit_off[u];
  int64_t* cursor = (int64_t*)malloc(sizeof(int64_t) * (size_t)U);
  memcpy(cursor, o->unit_off, sizeof(int64_t) * (size_t)U);
  uint64_t* keys = (uint64_t*)malloc(sizeof(uint64_t) * 2 * (size_t)(N > 0 ? N : 1));
  for (int64_t i = 0; i < N; i++) { int64_t p = cursor[all[i].unit]++; keys[2 * p] = mix64(mix64(P->seed ^ 0xABCDEF12345ULL) + (uint64_t)i); keys[2 * p + 1] = (uint64_t)i; }
  free(cursor);
#pragma omp parallel for schedule(dynamic, 16)
  for (int u = 0; u < U; u++) { int64_t a = o->unit_off[u], b = o->unit_off[u + 1]; if (b - a > 1) qsort(keys + 2 * a, (size_t)(b - a), 2 * sizeof(uint64_t), cmp_u64pair); }
  o->n_clusters = N;
  o->y = (float*)malloc(sizeof(float) * (size_t)(N + 1)); o->t = (float*)malloc(sizeof(float) * (size_t)(N + 1));
  o->q = (float*)malloc(sizeof(float) * (size_t)(N + 1)); o->label = (int32_t*)malloc(sizeof(int32_t) * (size_t)(N + 1));
  o->leg0 = (uint8_t*)malloc((size_t)(N + 1));
#pragma omp parallel for schedule(static)
  for (int64_t p = 0; p < N; p++) { const cl_t* c = &all[keys[2 * p + 1]];
    o->y[p] = c->y; o->t[p] = c->t; o->q[p] = c->q; o->label[p] = c->label; o->leg0[p] = c->leg0; }
  free(keys); free(all); free(parts); free(row_x);
  return 0;
}
