/* otoo_oracle.c -- see otoo_oracle.h.  TEST INFRASTRUCTURE ONLY; plain C99 + OpenMP.
 * Compile with -ffp-contract=off so that no a*b+c is fused behind our back; fmaf() is used
 * where DESIGN.md's readings state a fused operation.
 * Citations are PAPER.md line numbers (L..) and DESIGN.md readings (R..). */
#include "otoo_oracle.h"
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define MAXLEV 21

struct orc_tree {
  int64_t N;
  int n_crit;
  int key_order;  /* 0 Morton (R3), 1 Hilbert (R20) */
  int dist_kind;  /* 0 group AABB distance (R8), 1 the paper's exact minimum over the members (L163; R23),
                     2 minimum over the AABBs of the group's pieces between its coarsest key boundaries (R25) */
  int split_pieces; /* dist_kind 2: number of pieces K (8) */
  float lo[3], S;
  uint64_t* key;  /* sorted keys */
  uint32_t* perm; /* perm[s] = original index of sorted slot s */
  float* spos;    /* sorted (x,y,z,m) */
  int64_t ncell, cap, nleaf;
  int depth;
  orc_cell* cell; /* canonical order after build */
  double* MP;     /* 4*ncell: M, Px, Py, Pz (unnormalised first moment), R6 */
  double* cm;     /* 3*ncell fp64 centre of mass */
  float* com_m;   /* 4*ncell fp32 (cm, m) as the walk sees them */
  double* s;      /* distance CM - geometric centre, R7 */
  /* paper-style linked list (L49-L57, L135): node < N particle slot, node >= N cell N+id */
  int64_t* next;
  int64_t* more;
};

/* ---------------- Hilbert order (PAPER III-B step 2, L131: "we convert the Morton key into the Hilbert key")
 * The paper gives no algorithm; reading R20: the 3-D Hilbert curve in Skilling's transpose
 * form ("Programming the Hilbert curve", 2004), b = 21 bits per axis, x the most significant axis.  The
 * key is the bit interleave of the transformed coordinates, so its top 3l bits still name the level-l
 * octree cell: the tree holds the same cells as with Morton keys, visited in Hilbert order. */
static void hilbert_axes_to_transpose(uint32_t X[3], int b) {
  uint32_t M = 1u << (b - 1), P, Q, t;
  for (Q = M; Q > 1; Q >>= 1) {
    P = Q - 1;
    for (int i = 0; i < 3; i++) {
      if (X[i] & Q) X[0] ^= P;                                       /* invert the low bits of x */
      else { t = (X[0] ^ X[i]) & P; X[0] ^= t; X[i] ^= t; }          /* exchange the low bits of x and axis i */
    }
  }
  for (int i = 1; i < 3; i++) X[i] ^= X[i - 1];                      /* Gray encode */
  t = 0;
  for (Q = M; Q > 1; Q >>= 1) if (X[2] & Q) t ^= Q - 1;
  for (int i = 0; i < 3; i++) X[i] ^= t;
}
static void hilbert_transpose_to_axes(uint32_t X[3], int b) {
  uint32_t N = 2u << (b - 1), P, Q, t;
  t = X[2] >> 1;                                                     /* Gray decode */
  for (int i = 2; i > 0; i--) X[i] ^= X[i - 1];
  X[0] ^= t;
  for (Q = 2; Q != N; Q <<= 1) {
    P = Q - 1;
    for (int i = 2; i >= 0; i--) {
      if (X[i] & Q) X[0] ^= P;
      else { t = (X[0] ^ X[i]) & P; X[0] ^= t; X[i] ^= t; }
    }
  }
}
static uint64_t interleave3(const uint32_t q[3]) {
  uint64_t key = 0;
  for (int b = 0; b < MAXLEV; b++)
    key |= (uint64_t)((((q[0] >> b) & 1u) << 2) | (((q[1] >> b) & 1u) << 1) | ((q[2] >> b) & 1u)) << (3 * b);
  return key;
}
uint64_t orc_hilbert_key(const uint32_t q_in[3]) {   /* quantised coordinates (21 bits each) -> 63-bit Hilbert key */
  uint32_t X[3] = {q_in[0], q_in[1], q_in[2]};
  hilbert_axes_to_transpose(X, MAXLEV);
  return interleave3(X);
}
void orc_hilbert_coords(uint64_t key, uint32_t q[3]) {   /* the inverse */
  q[0] = q[1] = q[2] = 0;
  for (int b = 0; b < MAXLEV; b++) {
    uint64_t oct = (key >> (3 * b)) & 7u;
    q[0] |= (uint32_t)((oct >> 2) & 1u) << b; q[1] |= (uint32_t)((oct >> 1) & 1u) << b; q[2] |= (uint32_t)(oct & 1u) << b;
  }
  hilbert_transpose_to_axes(q, MAXLEV);
}

/* ---------------- R1-R4: root cube, keys, sort (PAPER III-B steps 1-3, L121-L133) --------- */
static uint64_t key_of_ord(const float lo[3], float scale, const float* p, int key_order) {
  uint32_t q[3];
  for (int k = 0; k < 3; k++) {
    float d = p[k] - lo[k];         /* one fp32 subtract */
    float t = d * scale;            /* one fp32 multiply */
    uint32_t v = (t >= 2097151.0f) ? 2097151u : (t > 0.0f ? (uint32_t)t : 0u);
    q[k] = v;
  }
  if (key_order == 1) return orc_hilbert_key(q);
  uint64_t key = 0;
  for (int lev = 1; lev <= MAXLEV; lev++) { /* L129: concatenation of the octant index per level */
    int b = MAXLEV - lev;
    uint64_t oct = (((q[0] >> b) & 1u) << 2) | (((q[1] >> b) & 1u) << 1) | ((q[2] >> b) & 1u);
    key |= oct << (3 * b);
  }
  return key;
}

typedef struct { uint64_t key; uint32_t id; } kv_t;
static int kv_cmp(const void* a, const void* b) {
  const kv_t* x = (const kv_t*)a; const kv_t* y = (const kv_t*)b;
  if (x->key != y->key) return x->key < y->key ? -1 : 1;
  if (x->id != y->id) return x->id < y->id ? -1 : 1;   /* R4: ties by original index */
  return 0;
}

static int64_t new_cell(orc_tree* t) {
  if (t->ncell == t->cap) {
    t->cap = t->cap ? 2 * t->cap : 1024;
    t->cell = (orc_cell*)realloc(t->cell, sizeof(orc_cell) * t->cap);
  }
  return t->ncell++;
}

/* R5 / L135: slice the sorted keys by octant index, recursively; leaf iff count <= n_crit or
 * level 21.  Cells are created in depth-first order here and renumbered afterwards. */
static void split(orc_tree* t, int64_t id) {
  orc_cell c = t->cell[id];
  if (c.count <= (uint32_t)t->n_crit || c.level == MAXLEV) { t->nleaf++; return; }
  int shift = 3 * (MAXLEV - (c.level + 1));
  int64_t kids[8]; int nk = 0;
  uint32_t s = c.first, end = c.first + c.count;
  while (s < end) {
    uint64_t oct = (t->key[s] >> shift) & 7u;
    uint32_t e = s;
    while (e < end && ((t->key[e] >> shift) & 7u) == oct) e++;
    int64_t k = new_cell(t);
    t->cell[k].prefix = t->key[s] >> shift;
    t->cell[k].first = s; t->cell[k].count = e - s;
    t->cell[k].level = (uint8_t)(c.level + 1);
    t->cell[k].child_first = 0; t->cell[k].child_count = 0;
    kids[nk++] = k;
    s = e;
  }
  t->cell[id].child_first = (uint32_t)kids[0];   /* the nk children were created consecutively */
  t->cell[id].child_count = (uint8_t)nk;
  for (int i = 0; i < nk; i++) split(t, kids[i]);
}

typedef struct { orc_cell c; int64_t old; } cs_t;
static int cs_cmp(const void* a, const void* b) {
  const cs_t* x = (const cs_t*)a; const cs_t* y = (const cs_t*)b;
  if (x->c.level != y->c.level) return x->c.level < y->c.level ? -1 : 1;
  if (x->c.first != y->c.first) return x->c.first < y->c.first ? -1 : 1;
  return 0;
}

static void cell_coord_ord(uint64_t prefix, int level, uint32_t c[3], int key_order) {
  if (key_order == 1) {   /* Hilbert prefix -> any key of the cell -> coordinates -> their top `level` bits */
    uint32_t q[3];
    if (level == 0) { c[0] = c[1] = c[2] = 0; return; }
    orc_hilbert_coords(prefix << (3 * (MAXLEV - level)), q);
    for (int k = 0; k < 3; k++) c[k] = q[k] >> (MAXLEV - level);
    return;
  }
  c[0] = c[1] = c[2] = 0;
  for (int i = 0; i < level; i++) {
    uint64_t oct = (prefix >> (3 * i)) & 7u;
    c[0] |= (uint32_t)((oct >> 2) & 1u) << i;
    c[1] |= (uint32_t)((oct >> 1) & 1u) << i;
    c[2] |= (uint32_t)(oct & 1u) << i;
  }
}

/* R6 / L155: recursive depth-first mass and first moment, fp64, fixed order. */
static void moments(orc_tree* t, int64_t id) {
  orc_cell* c = &t->cell[id];
  double M = 0, Px = 0, Py = 0, Pz = 0;
  if (c->child_count == 0) {
    for (uint32_t s = c->first; s < c->first + c->count; s++) {
      const float* p = t->spos + 4 * (int64_t)s;
      double m = p[3];
      M = M + m;
      Px = Px + m * (double)p[0];
      Py = Py + m * (double)p[1];
      Pz = Pz + m * (double)p[2];
    }
  } else {
    for (int k = 0; k < c->child_count; k++) {
      int64_t ch = (int64_t)c->child_first + k;
      moments(t, ch);
      M = M + t->MP[4 * ch];
      Px = Px + t->MP[4 * ch + 1];
      Py = Py + t->MP[4 * ch + 2];
      Pz = Pz + t->MP[4 * ch + 3];
    }
  }
  t->MP[4 * id] = M; t->MP[4 * id + 1] = Px; t->MP[4 * id + 2] = Py; t->MP[4 * id + 3] = Pz;
  /* geometric centre and s (R7) */
  uint32_t cc[3]; cell_coord_ord(c->prefix, c->level, cc, t->key_order);
  double l = ldexp((double)t->S, -(int)c->level);
  double g[3];
  for (int k = 0; k < 3; k++) g[k] = (double)t->lo[k] + ((double)cc[k] + 0.5) * l;
  double cm[3];
  if (M != 0.0) { cm[0] = Px / M; cm[1] = Py / M; cm[2] = Pz / M; }
  else { cm[0] = g[0]; cm[1] = g[1]; cm[2] = g[2]; }
  for (int k = 0; k < 3; k++) { t->cm[3 * id + k] = cm[k]; t->com_m[4 * id + k] = (float)cm[k]; }
  t->com_m[4 * id + 3] = (float)M;
  double dx = cm[0] - g[0], dy = cm[1] - g[1], dz = cm[2] - g[2];
  t->s[id] = sqrt((dx * dx + dy * dy) + dz * dz);
}

orc_tree* orc_build(int64_t N, const float* pos_mass, int n_crit) { return orc_build_ord(N, pos_mass, n_crit, 0); }
orc_tree* orc_build_ord(int64_t N, const float* pos_mass, int n_crit, int key_order) {
  orc_tree* t = (orc_tree*)calloc(1, sizeof(orc_tree));
  t->N = N; t->n_crit = n_crit; t->key_order = key_order;
  t->dist_kind = 2; t->split_pieces = 8;   /* R25 is the default group-cell distance of the gravity walks */
  /* R1 / L121,L127: cube enclosing all particles, anchored at the lo corner */
  float lo[3] = {0, 0, 0}, hi[3] = {0, 0, 0};
  for (int64_t i = 0; i < N; i++)
    for (int k = 0; k < 3; k++) {
      float v = pos_mass[4 * i + k];
      if (i == 0 || v < lo[k]) lo[k] = v;
      if (i == 0 || v > hi[k]) hi[k] = v;
    }
  float S = 0.0f;
  for (int k = 0; k < 3; k++) { float d = hi[k] - lo[k]; if (d > S) S = d; t->lo[k] = lo[k]; }
  if (!(S > 0.0f)) S = 1.0f;
  t->S = S;
  float scale = 2097152.0f / S;   /* R2: IEEE fp32 division */
  kv_t* kv = (kv_t*)malloc(sizeof(kv_t) * (N > 0 ? N : 1));
#pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < N; i++) { kv[i].key = key_of_ord(lo, scale, pos_mass + 4 * i, key_order); kv[i].id = (uint32_t)i; }
  qsort(kv, (size_t)N, sizeof(kv_t), kv_cmp);   /* L133 */
  t->key = (uint64_t*)malloc(8 * (N > 0 ? N : 1));
  t->perm = (uint32_t*)malloc(4 * (N > 0 ? N : 1));
  t->spos = (float*)malloc(16 * (N > 0 ? N : 1));
  for (int64_t s = 0; s < N; s++) {
    t->key[s] = kv[s].key; t->perm[s] = kv[s].id;
    memcpy(t->spos + 4 * s, pos_mass + 4 * (int64_t)kv[s].id, 16);
  }
  free(kv);
  /* R5: topology */
  int64_t root = new_cell(t);
  t->cell[root].prefix = 0; t->cell[root].first = 0; t->cell[root].count = (uint32_t)N;
  t->cell[root].level = 0; t->cell[root].child_first = 0; t->cell[root].child_count = 0;
  split(t, root);
  /* canonical renumbering: level ascending, then first ascending */
  cs_t* cs = (cs_t*)malloc(sizeof(cs_t) * t->ncell);
  for (int64_t i = 0; i < t->ncell; i++) { cs[i].c = t->cell[i]; cs[i].old = i; }
  qsort(cs, (size_t)t->ncell, sizeof(cs_t), cs_cmp);
  int64_t* newid = (int64_t*)malloc(8 * t->ncell);
  for (int64_t i = 0; i < t->ncell; i++) newid[cs[i].old] = i;
  t->depth = 0;
  for (int64_t i = 0; i < t->ncell; i++) {
    t->cell[i] = cs[i].c;
    if (t->cell[i].child_count) t->cell[i].child_first = (uint32_t)newid[cs[i].c.child_first];
    if (t->cell[i].level > t->depth) t->depth = t->cell[i].level;
  }
  free(cs); free(newid);
  /* R6, R7 */
  t->MP = (double*)malloc(32 * t->ncell);
  t->cm = (double*)malloc(24 * t->ncell);
  t->com_m = (float*)malloc(16 * t->ncell);
  t->s = (double*)malloc(8 * t->ncell);
  moments(t, 0);
  /* L49-L57, L135: next/more linked list, particles 0..N-1, cells N.. */
  t->next = (int64_t*)malloc(8 * (N + t->ncell));
  t->more = (int64_t*)malloc(8 * (N + t->ncell));
  for (int64_t i = 0; i < N; i++) t->more[i] = -1;
  t->next[N + 0] = -1;
  for (int64_t id = 0; id < t->ncell; id++) {   /* parents precede children in canonical order */
    orc_cell* c = &t->cell[id];
    int64_t after = t->next[N + id];
    if (c->child_count == 0) {
      if (c->count == 0) { t->more[N + id] = after; continue; }
      t->more[N + id] = c->first;
      for (uint32_t s = c->first; s < c->first + c->count; s++)
        t->next[s] = (s + 1 < c->first + c->count) ? (int64_t)(s + 1) : after;
    } else {
      t->more[N + id] = N + c->child_first;
      for (int k = 0; k < c->child_count; k++)
        t->next[N + c->child_first + k] = (k + 1 < c->child_count) ? N + c->child_first + k + 1 : after;
    }
  }
  return t;
}

void orc_free(orc_tree* t) {
  if (!t) return;
  free(t->key); free(t->perm); free(t->spos); free(t->cell); free(t->MP); free(t->cm);
  free(t->com_m); free(t->s); free(t->next); free(t->more); free(t);
}
int64_t orc_ncell(const orc_tree* t) { return t->ncell; }
int64_t orc_nleaf(const orc_tree* t) { return t->nleaf; }
int orc_depth(const orc_tree* t) { return t->depth; }
void orc_root(const orc_tree* t, float lo[3], float* S) { memcpy(lo, t->lo, 12); *S = t->S; }
uint64_t orc_key(const orc_tree* t, const float xyz[3]) { return key_of_ord(t->lo, 2097152.0f / t->S, xyz, t->key_order); }

void orc_export(const orc_tree* t, uint32_t* perm, uint64_t* keys, orc_cell* cells, float* com_m,
                double* s, double* MP) {
  if (perm) memcpy(perm, t->perm, 4 * t->N);
  if (keys) memcpy(keys, t->key, 8 * t->N);
  if (cells) memcpy(cells, t->cell, sizeof(orc_cell) * t->ncell);
  if (com_m) memcpy(com_m, t->com_m, 16 * t->ncell);
  if (s) memcpy(s, t->s, 8 * t->ncell);
  if (MP) memcpy(MP, t->MP, 32 * t->ncell);
}

/* ---------------- direct sum: the plain O(N^2) definition (L43 "O(N^2) ... brute force") ----- */
void orc_direct_sum(int64_t N, const float* pm, double eps, int64_t nt, const int64_t* targets,
                    double* out) {
  int64_t T = targets ? nt : N;
  double e2 = eps * eps;
#pragma omp parallel for schedule(dynamic, 16)
  for (int64_t t = 0; t < T; t++) {
    int64_t i = targets ? targets[t] : t;
    double xi = pm[4 * i], yi = pm[4 * i + 1], zi = pm[4 * i + 2];
    double ax = 0, ay = 0, az = 0, ph = 0;
    for (int64_t j = 0; j < N; j++) {
      if (j == i) continue;
      double dx = (double)pm[4 * j] - xi, dy = (double)pm[4 * j + 1] - yi, dz = (double)pm[4 * j + 2] - zi;
      double r2 = dx * dx + dy * dy + dz * dz + e2;
      if (r2 == 0.0) continue;
      double ri = 1.0 / sqrt(r2);
      double m = pm[4 * j + 3];
      double mr3 = m * ri * ri * ri;
      ax += mr3 * dx; ay += mr3 * dy; az += mr3 * dz; ph -= m * ri;
    }
    out[4 * t] = ax; out[4 * t + 1] = ay; out[4 * t + 2] = az; out[4 * t + 3] = ph;
  }
}

/* ---------------- R7: theta-MAC bounding radius (the paper's r_b abstraction, L61) ---------- */
void orc_rb2(const orc_tree* t, double theta, int mac_kind, float* rb2) {
  for (int64_t id = 0; id < t->ncell; id++) {
    if (theta <= 0.0) { rb2[id] = INFINITY; continue; }
    double l = ldexp((double)t->S, -(int)t->cell[id].level);
    double rb = l / theta;
    if (mac_kind == 0) rb = rb + t->s[id];
    rb2[id] = (float)(rb * rb);
  }
}

/* ---------------- the paper's own MAC: absolute-error criterion (PAPER II-B Eq. 1-2; III-C L157)
 * B2 (Eq. 2) = sum over the cell's particles of m |r_CM - r|^2.  Reading R19: like mass and
 * centre of mass (R6) it is accumulated bottom-up in a fixed order so that it is reproducible bit for bit:
 * leaf: sequentially over its particles in sorted order; internal cell: over its children in octant order
 * with the parallel-axis theorem, B2 += B2_child, then B2 += M_child |CM_child - CM|^2.  orc_B2_direct is
 * Eq. 2 written out (the pin).  b_max = max over ALL particles of the cell of |r - CM| (fp64, L63). */
void orc_delta_cell_props(const orc_tree* t, double* B2, double* bmax) {
  for (int64_t id = t->ncell - 1; id >= 0; id--) {   /* canonical ids: children come after their parent */
    const orc_cell* c = &t->cell[id];
    const double* cm = t->cm + 3 * id;
    double b2 = 0.0;
    if (c->child_count == 0) {
      for (uint32_t s = c->first; s < c->first + c->count; s++) {
        const float* p = t->spos + 4 * (int64_t)s;
        double dx = (double)p[0] - cm[0], dy = (double)p[1] - cm[1], dz = (double)p[2] - cm[2];
        double r2 = (dx * dx + dy * dy) + dz * dz;
        b2 = b2 + (double)p[3] * r2;
      }
    } else {
      for (int k = 0; k < c->child_count; k++) {
        int64_t ch = (int64_t)c->child_first + k;
        const double* cc = t->cm + 3 * ch;
        double dx = cc[0] - cm[0], dy = cc[1] - cm[1], dz = cc[2] - cm[2];
        double r2 = (dx * dx + dy * dy) + dz * dz;
        b2 = b2 + B2[ch];
        b2 = b2 + t->MP[4 * ch] * r2;
      }
    }
    B2[id] = b2;
    if (bmax) {
      double b = 0.0;
      for (uint32_t s = c->first; s < c->first + c->count; s++) {
        const float* p = t->spos + 4 * (int64_t)s;
        double dx = (double)p[0] - cm[0], dy = (double)p[1] - cm[1], dz = (double)p[2] - cm[2];
        double r = sqrt((dx * dx + dy * dy) + dz * dz);
        if (r > b) b = r;
      }
      bmax[id] = b;
    }
  }
}
double orc_B2_direct(const orc_tree* t, int64_t id) {   /* Eq. 2 as printed */
  const orc_cell* c = &t->cell[id];
  const double* cm = t->cm + 3 * id;
  double b2 = 0.0;
  for (uint32_t s = c->first; s < c->first + c->count; s++) {
    const float* p = t->spos + 4 * (int64_t)s;
    double dx = cm[0] - (double)p[0], dy = cm[1] - (double)p[1], dz = cm[2] - (double)p[2];
    b2 += (double)p[3] * (dx * dx + dy * dy + dz * dz);
  }
  return b2;
}
/* Eq. 1: r_b = b/2 + sqrt(b^2/4 + sqrt(3 B2 / Delta)); cells heavier than m_limit: r_b = 2 S_root (L157);
 * Delta <= 0: open everything.  rb^2 rounded once to fp32, as for the theta-MAC (R7). */
void orc_rb2_delta(const orc_tree* t, double delta, double m_limit, float* rb2) {
  double* B2 = (double*)malloc(8 * t->ncell);
  double* bm = (double*)malloc(8 * t->ncell);
  orc_delta_cell_props(t, B2, bm);
  for (int64_t id = 0; id < t->ncell; id++) {
    double rb;
    if (!(delta > 0.0)) { rb2[id] = INFINITY; continue; }
    if (t->MP[4 * id] > m_limit) rb = 2.0 * (double)t->S;
    else {
      double h = 0.5 * bm[id];
      double q = sqrt((3.0 * B2[id]) / delta);
      rb = h + sqrt(h * h + q);
    }
    rb2[id] = (float)(rb * rb);
  }
  free(B2); free(bm);
}

/* ---------------- R8: group AABB and group-cell distance (L163, Barnes 1990 form) ----------- */
#define MAXPIECES 16
typedef struct {
  float lo[3], hi[3]; float hmax; const float* mem; int nmem;   /* mem: the members' (x,y,z,m), set for dist_kind 1 */
  int npiece; float plo[MAXPIECES][3], phi[MAXPIECES][3];       /* dist_kind 2: tight boxes of the pieces */
  float phmax[MAXPIECES];                                       /* SPH: largest h of each piece */
} gbox_t;
static int key_cplev(uint64_t a, uint64_t b) {   /* number of leading octree levels two keys share, 0..21 */
  int l = 0;
  while (l < MAXLEV && ((a >> (3 * (MAXLEV - 1 - l))) & 7u) == ((b >> (3 * (MAXLEV - 1 - l))) & 7u)) l++;
  return l;
}
/* Reading R25: the group [a, b) is cut at its K-1 coarsest key boundaries -- the slots s in (a, b) with
 * the smallest number of octree levels shared by key[s-1] and key[s] (ties: the lowest slot first).  A Morton
 * range that crosses the boundary of a coarse cell jumps across that cell (the curve is not continuous), so the
 * bounding box of the whole group can be as large as the cell while each piece between two such boundaries is
 * compact.  The group-cell distance is the minimum over the pieces of the box distance of R8. */
static void split_pieces(const orc_tree* t, int64_t a, int64_t b, int K, gbox_t* g, const float* hs) {
  int64_t cut[MAXPIECES]; int ncut = 0;
  int n = (int)(b - a);
  if (K > MAXPIECES) K = MAXPIECES;
  unsigned char* taken = (unsigned char*)calloc(n > 0 ? n : 1, 1);
  for (int k = 0; k < K - 1 && k < n - 1; k++) {          /* the k-th coarsest boundary */
    int best = -1, bl = MAXLEV + 1;
    for (int i = 1; i < n; i++) {
      if (taken[i]) continue;
      int l = key_cplev(t->key[a + i - 1], t->key[a + i]);
      if (l < bl) { bl = l; best = i; }                   /* strict: ties keep the lowest slot */
    }
    taken[best] = 1;
  }
  for (int i = 1; i < n; i++) if (taken[i]) cut[ncut++] = a + i;   /* in slot order */
  free(taken);
  g->npiece = ncut + 1;
  for (int p = 0; p <= ncut; p++) {
    int64_t s0 = p == 0 ? a : cut[p - 1], s1 = p == ncut ? b : cut[p];
    for (int k = 0; k < 3; k++) { g->plo[p][k] = t->spos[4 * s0 + k]; g->phi[p][k] = g->plo[p][k]; }
    g->phmax[p] = 0.0f;
    for (int64_t s = s0; s < s1; s++) {
      for (int k = 0; k < 3; k++) {
        float v = t->spos[4 * s + k];
        if (v < g->plo[p][k]) g->plo[p][k] = v;
        if (v > g->phi[p][k]) g->phi[p][k] = v;
      }
      if (hs && hs[s] > g->phmax[p]) g->phmax[p] = hs[s];
    }
  }
}
static gbox_t group_box(const orc_tree* t, int64_t a, int64_t b, const float* hs /*sorted h or NULL*/) {
  gbox_t g; g.hmax = 0.0f; g.npiece = 0;
  g.mem = (t->dist_kind == 1 && !hs) ? t->spos + 4 * a : NULL; g.nmem = (int)(b - a);   /* SPH walks (hs given) have no exact-minimum form: one box */
  if (t->dist_kind == 2 && !hs) split_pieces(t, a, b, t->split_pieces, &g, NULL);
  if (hs && t->dist_kind == 2) split_pieces(t, a, b, t->split_pieces, &g, hs);   /* SPH walks: R26 */
  for (int k = 0; k < 3; k++) { g.lo[k] = t->spos[4 * a + k]; g.hi[k] = g.lo[k]; }
  for (int64_t s = a; s < b; s++) {
    for (int k = 0; k < 3; k++) {
      float v = t->spos[4 * s + k];
      if (v < g.lo[k]) g.lo[k] = v;
      if (v > g.hi[k]) g.hi[k] = v;
    }
    if (hs && hs[s] > g.hmax) g.hmax = hs[s];
  }
  return g;
}
static float box_d2(const gbox_t* g, const float* cm) {
  if (g->mem) {
    /* "compute n_vec distances for each pair and then select the actual minimum distance";
     * reading R23: d_i^2 = fma(dz,dz, fma(dy,dy, dx*dx)), d = fl32(x_i - cm), in fp32; the minimum is exact */
    float best = INFINITY;
    for (int i = 0; i < g->nmem; i++) {
      float dx = g->mem[4 * i] - cm[0], dy = g->mem[4 * i + 1] - cm[1], dz = g->mem[4 * i + 2] - cm[2];
      float d2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
      if (d2 < best) best = d2;
    }
    return best;
  }
  if (g->npiece > 0) {   /* R25: minimum over the pieces' boxes of the R8 expression (the minimum of fp32 values is exact) */
    float best = INFINITY;
    for (int p = 0; p < g->npiece; p++) {
      float e[3];
      for (int k = 0; k < 3; k++) {
        float a = g->plo[p][k] - cm[k], b = cm[k] - g->phi[p][k];
        float m = a > b ? a : b;
        e[k] = m > 0.0f ? m : 0.0f;
      }
      float d2 = fmaf(e[2], e[2], fmaf(e[1], e[1], e[0] * e[0]));
      if (d2 < best) best = d2;
    }
    return best;
  }
  float e[3];
  for (int k = 0; k < 3; k++) {
    float a = g->lo[k] - cm[k], b = cm[k] - g->hi[k];
    float m = a > b ? a : b;
    e[k] = m > 0.0f ? m : 0.0f;
  }
  return fmaf(e[2], e[2], fmaf(e[1], e[1], e[0] * e[0]));
}

typedef struct {
  uint32_t *cells, *parts; int64_t nc, np, capc, capp; uint32_t ntests;
} lists_t;
static void push_u32(uint32_t** a, int64_t* n, int64_t* cap, uint32_t v) {
  if (*n == *cap) { *cap = *cap ? 2 * *cap : 4096; *a = (uint32_t*)realloc(*a, 4 * *cap); }
  (*a)[(*n)++] = v;
}

/* R9 / L57 rules as a recursion: accepted -> cell list; not accepted leaf -> its particles;
 * otherwise descend.  Particles are never MAC-tested (rule 3). */
static void walk_rec(const orc_tree* t, const float* rb2, const gbox_t* g, int64_t id, lists_t* L) {
  const orc_cell* c = &t->cell[id];
  L->ntests++;
  float d2 = box_d2(g, t->com_m + 4 * id);
  if (d2 > rb2[id]) { push_u32(&L->cells, &L->nc, &L->capc, (uint32_t)id); return; }
  if (c->child_count == 0) {
    for (uint32_t s = c->first; s < c->first + c->count; s++) push_u32(&L->parts, &L->np, &L->capp, s);
    return;
  }
  for (int k = 0; k < c->child_count; k++) walk_rec(t, rb2, g, (int64_t)c->child_first + k, L);
}
/* The paper's own iterative traversal, literally (L57 rules 1-4). */
static void walk_stackless(const orc_tree* t, const float* rb2, const gbox_t* g, lists_t* L) {
  int64_t N = t->N, node = N;                       /* start from the root cell */
  while (node != -1) {                              /* (4) null pointer: stop */
    if (node < N) {                                 /* (3) particle: interact, follow next */
      push_u32(&L->parts, &L->np, &L->capp, (uint32_t)node);
      node = t->next[node];
    } else {
      int64_t id = node - N;
      L->ntests++;
      float d2 = box_d2(g, t->com_m + 4 * id);
      if (d2 > rb2[id]) {                           /* (2) accepted: interact, follow next */
        push_u32(&L->cells, &L->nc, &L->capc, (uint32_t)id);
        node = t->next[node];
      } else node = t->more[node];                  /* (1) not accepted: follow more */
    }
  }
}

/* R10: softened Plummer sums, fp64, with the fp32-rounded cell data the walk uses. */
static void grav_sums(const orc_tree* t, const lists_t* L, int64_t slot, double e2, double* out, double* abs_out) {
  const float* p = t->spos + 4 * slot;
  double xi = p[0], yi = p[1], zi = p[2];
  double ax = 0, ay = 0, az = 0, ph = 0, asum = 0;
  for (int64_t k = 0; k < L->nc; k++) {
    const float* c = t->com_m + 4 * (int64_t)L->cells[k];
    double dx = (double)c[0] - xi, dy = (double)c[1] - yi, dz = (double)c[2] - zi;
    double r2 = dx * dx + dy * dy + dz * dz + e2;
    if (r2 == 0.0) continue;
    double ri = 1.0 / sqrt(r2), m = c[3];
    double mr3 = m * ri * ri * ri;
    ax += mr3 * dx; ay += mr3 * dy; az += mr3 * dz; ph -= m * ri;
    asum += mr3 * sqrt(dx * dx + dy * dy + dz * dz);   /* |a_ij|, for the test's error bound */
  }
  for (int64_t k = 0; k < L->np; k++) {
    int64_t j = L->parts[k];
    if (j == slot) continue;                        /* self term excluded by index */
    const float* q = t->spos + 4 * j;
    double dx = (double)q[0] - xi, dy = (double)q[1] - yi, dz = (double)q[2] - zi;
    double r2 = dx * dx + dy * dy + dz * dz + e2;
    if (r2 == 0.0) continue;
    double ri = 1.0 / sqrt(r2), m = q[3];
    double mr3 = m * ri * ri * ri;
    ax += mr3 * dx; ay += mr3 * dy; az += mr3 * dz; ph -= m * ri;
    asum += mr3 * sqrt(dx * dx + dy * dy + dz * dz);   /* |a_ij|, for the test's error bound */
  }
  out[0] = ax; out[1] = ay; out[2] = az; out[3] = ph;
  if (abs_out) *abs_out = asum;
}

/* sel != NULL: only the groups sel[0..nsel) are walked (counters indexed by position in sel, sums written
 * for their targets only); the loop over groups is then serial and the targets of a group run in parallel,
 * so that one system-sized group does not serialise the run.  Same arithmetic either way. */
uint64_t orc_gravity_rb2(const orc_tree* t, double eps, const float* rb2, int G, int walk_kind,
                         const int64_t* sel, int64_t nsel,
                         double* acc_pot, uint32_t* n_tests, uint32_t* n_cells, uint32_t* n_parts, double* abs_sum) {
  int64_t N = t->N, ng = sel ? nsel : (N + G - 1) / G;
  double e2 = eps * eps;
  uint64_t total = 0;
#pragma omp parallel reduction(+ : total) if (sel == NULL)
  {
    lists_t L; memset(&L, 0, sizeof L);
#pragma omp for schedule(dynamic, 1)
    for (int64_t gi = 0; gi < ng; gi++) {
      int64_t g = sel ? sel[gi] : gi;
      int64_t a = g * G, b = a + G < N ? a + G : N;
      gbox_t box = group_box(t, a, b, NULL);
      L.nc = L.np = 0; L.ntests = 0;
      if (walk_kind == 0) walk_rec(t, rb2, &box, 0, &L); else walk_stackless(t, rb2, &box, &L);
      if (n_tests) n_tests[gi] = L.ntests;
      if (n_cells) n_cells[gi] = (uint32_t)L.nc;
      if (n_parts) n_parts[gi] = (uint32_t)L.np;
      total += (uint64_t)(b - a) * (uint64_t)(L.nc + L.np);   /* R11 */
      if (acc_pot) {
#pragma omp parallel for schedule(dynamic, 1) if (sel != NULL)
        for (int64_t s = a; s < b; s++)
          grav_sums(t, &L, s, e2, acc_pot + 4 * (int64_t)t->perm[s], abs_sum ? abs_sum + t->perm[s] : NULL);
      }
    }
    free(L.cells); free(L.parts);
  }
  return total;
}
uint64_t orc_gravity_sel(const orc_tree* t, double eps, double theta, int G, int mac_kind, int walk_kind,
                         const int64_t* sel, int64_t nsel,
                         double* acc_pot, uint32_t* n_tests, uint32_t* n_cells, uint32_t* n_parts, double* abs_sum) {
  float* rb2 = (float*)malloc(4 * t->ncell);
  orc_rb2(t, theta, mac_kind, rb2);
  uint64_t total = orc_gravity_rb2(t, eps, rb2, G, walk_kind, sel, nsel, acc_pot, n_tests, n_cells, n_parts, abs_sum);
  free(rb2);
  return total;
}
uint64_t orc_gravity(const orc_tree* t, double eps, double theta, int G, int mac_kind, int walk_kind,
                     double* acc_pot, uint32_t* n_tests, uint32_t* n_cells, uint32_t* n_parts, double* abs_sum) {
  return orc_gravity_sel(t, eps, theta, G, mac_kind, walk_kind, NULL, 0, acc_pot, n_tests, n_cells, n_parts, abs_sum);
}

void orc_group_lists_rb2(const orc_tree* t, const float* rb2, int G, int64_t g,
                         uint32_t* cell_ids, uint32_t* part_slots) {
  int64_t a = g * G, b = a + G < t->N ? a + G : t->N;
  gbox_t box = group_box(t, a, b, NULL);
  lists_t L; memset(&L, 0, sizeof L);
  walk_rec(t, rb2, &box, 0, &L);
  if (cell_ids) memcpy(cell_ids, L.cells, 4 * L.nc);
  if (part_slots) memcpy(part_slots, L.parts, 4 * L.np);
  free(L.cells); free(L.parts);
}
void orc_group_lists(const orc_tree* t, double theta, int G, int mac_kind, int64_t g,
                     uint32_t* cell_ids, uint32_t* part_slots) {
  float* rb2 = (float*)malloc(4 * t->ncell);
  orc_rb2(t, theta, mac_kind, rb2);
  orc_group_lists_rb2(t, rb2, G, g, cell_ids, part_slots);
  free(rb2);
}

/* ---------------- SPH (PAPER II-C, L85-L105; readings R13-R17) ------------------------------ */
/* R13: cubic spline, h = support radius (L89: W "is zero outside of a given neighbor radius h") */
double orc_W(double r, double h) {
  double q = r / h, sig = 8.0 / (M_PI * h * h * h);
  if (q <= 0.5) return sig * (1.0 - 6.0 * q * q + 6.0 * q * q * q);
  if (q < 1.0) { double u = 1.0 - q; return sig * 2.0 * u * u * u; }
  return 0.0;
}
double orc_dWdr(double r, double h) {
  double q = r / h, sig = 8.0 / (M_PI * h * h * h * h);
  if (q <= 0.5) return sig * (-12.0 * q + 18.0 * q * q);
  if (q < 1.0) { double u = 1.0 - q; return sig * (-6.0 * u * u); }
  return 0.0;
}

static float* sorted_h(const orc_tree* t, const float* h) {
  float* hs = (float*)malloc(4 * (t->N > 0 ? t->N : 1));
  for (int64_t s = 0; s < t->N; s++) hs[s] = h[t->perm[s]];
  return hs;
}
static float up32(double v) { /* fp32 rounded up (R14) */
  float f = (float)v;
  if ((double)f < v) f = nextafterf(f, INFINITY);
  return f;
}
/* R14 / Eq. 5 (L101-L105): per cell, over ALL particles of the cell, from the fp64 CM. */
static void sph_radii_sorted(const orc_tree* t, const float* hs, float* bmax, float* rsph) {
#pragma omp parallel for schedule(dynamic, 64)
  for (int64_t id = 0; id < t->ncell; id++) {
    const orc_cell* c = &t->cell[id];
    double b = 0.0, r = 0.0;
    for (uint32_t s = c->first; s < c->first + c->count; s++) {
      const float* p = t->spos + 4 * (int64_t)s;
      double dx = (double)p[0] - t->cm[3 * id], dy = (double)p[1] - t->cm[3 * id + 1], dz = (double)p[2] - t->cm[3 * id + 2];
      double d = sqrt((dx * dx + dy * dy) + dz * dz);
      if (d > b) b = d;
      double dh = d + (double)hs[s];
      if (dh > r) r = dh;
    }
    bmax[id] = up32(b); rsph[id] = up32(r);
  }
}
void orc_sph_cell_radii(const orc_tree* t, const float* h, float* bmax, float* rsph) {
  float* hs = sorted_h(t, h);
  sph_radii_sorted(t, hs, bmax, rsph);
  free(hs);
}

/* R15: open iff d^2 <= R^2, R = max(r_SPH, b_max + h_max,g); no cell list (L105). */
static void walk_sph(const orc_tree* t, const float* bmax, const float* rsph, const gbox_t* g,
                     int64_t id, lists_t* L) {
  const orc_cell* c = &t->cell[id];
  L->ntests++;
  if (g->npiece > 0) {
    /* R26: the cell is opened iff SOME piece p of the group has d_p^2 <= R_p^2, d_p = box distance of the piece (R8
     * expression), R_p = max(r_SPH, b_max + h_max of the piece): the R15 test per piece */
    int open = 0;
    const float* cm = t->com_m + 4 * id;
    for (int p = 0; p < g->npiece && !open; p++) {
      float e[3];
      for (int k = 0; k < 3; k++) {
        float a = g->plo[p][k] - cm[k], b = cm[k] - g->phi[p][k];
        float m = a > b ? a : b;
        e[k] = m > 0.0f ? m : 0.0f;
      }
      float d2 = fmaf(e[2], e[2], fmaf(e[1], e[1], e[0] * e[0]));
      float R = fmaxf(rsph[id], bmax[id] + g->phmax[p]);
      if (d2 <= R * R) open = 1;
    }
    if (!open) return;
  } else {
    float d2 = box_d2(g, t->com_m + 4 * id);
    float R = fmaxf(rsph[id], bmax[id] + g->hmax);
    float R2 = R * R;
    if (!(d2 <= R2)) return;
  }
  if (c->child_count == 0) {
    for (uint32_t s = c->first; s < c->first + c->count; s++) push_u32(&L->parts, &L->np, &L->capp, s);
    return;
  }
  for (int k = 0; k < c->child_count; k++) walk_sph(t, bmax, rsph, g, (int64_t)c->child_first + k, L);
}
static float r2_f32(const float* a, const float* b) { /* R16: the fp32 neighbour distance */
  float dx = b[0] - a[0], dy = b[1] - a[1], dz = b[2] - a[2];
  return fmaf(dz, dz, fmaf(dy, dy, dx * dx));
}

uint64_t orc_sph_density_sel(const orc_tree* t, const float* h, int G, const int64_t* sel, int64_t nsel,
                             double* rho, uint32_t* nngb, uint32_t* n_tests, uint32_t* n_parts) {
  int64_t N = t->N, ng = sel ? nsel : (N + G - 1) / G;
  float* hs = sorted_h(t, h);
  float* bmax = (float*)malloc(4 * t->ncell); float* rsph = (float*)malloc(4 * t->ncell);
  sph_radii_sorted(t, hs, bmax, rsph);
  uint64_t total = 0;
#pragma omp parallel reduction(+ : total)
  {
    lists_t L; memset(&L, 0, sizeof L);
#pragma omp for schedule(dynamic, 1)
    for (int64_t gi = 0; gi < ng; gi++) {
      int64_t g = sel ? sel[gi] : gi;
      int64_t a = g * G, b = a + G < N ? a + G : N;
      gbox_t box = group_box(t, a, b, hs);
      L.np = 0; L.ntests = 0;
      walk_sph(t, bmax, rsph, &box, 0, &L);
      if (n_tests) n_tests[gi] = L.ntests;
      if (n_parts) n_parts[gi] = (uint32_t)L.np;
      total += (uint64_t)(b - a) * (uint64_t)L.np;
      for (int64_t s = a; s < b && rho; s++) {
        const float* pi = t->spos + 4 * s;
        float hi = hs[s], h2 = hi * hi;
        double sum = 0.0; uint32_t cnt = 0;
        for (int64_t k = 0; k < L.np; k++) {
          const float* pj = t->spos + 4 * (int64_t)L.parts[k];
          if (!(r2_f32(pi, pj) < h2)) continue;      /* R16: decision in fp32 */
          double dx = (double)pj[0] - pi[0], dy = (double)pj[1] - pi[1], dz = (double)pj[2] - pi[2];
          double r = sqrt(dx * dx + dy * dy + dz * dz);
          sum += (double)pj[3] * orc_W(r, (double)hi);   /* Eq. 4 (L87) with A = m */
          cnt++;
        }
        rho[t->perm[s]] = sum;
        if (nngb) nngb[t->perm[s]] = cnt;
      }
    }
    free(L.parts); free(L.cells);
  }
  free(hs); free(bmax); free(rsph);
  return total;
}

uint64_t orc_sph_density(const orc_tree* t, const float* h, int G, double* rho, uint32_t* nngb,
                         uint32_t* n_tests, uint32_t* n_parts) {
  return orc_sph_density_sel(t, h, G, NULL, 0, rho, nngb, n_tests, n_parts);
}
/* ---------------- SPH stage 1 with velocity derivatives (PAPER L252 step 4: "density, div v, rot v").  The paper
 * prints no formula; reading R22: the standard gather estimates with the particle's own h,
 *   div v_i = (1/rho_i) sum_j m_j (v_j - v_i) . grad_i W(r_ij, h_i)
 *   rot v_i = (1/rho_i) sum_j m_j (v_i - v_j) x grad_i W(r_ij, h_i),   grad_i W = dW/dr (x_i - x_j)/r,
 * over the neighbours of R16 (fp32 decision r^2 < h_i^2), r > 0, with rho_i of R16 (from the same pass).
 * out: 4N doubles (div, rot_x, rot_y, rot_z), caller's order; abs_sum (N or NULL): sum_j m_j |v_j - v_i| |dW/dr| / rho_i. */
uint64_t orc_sph_divrot_sel(const orc_tree* t, const float* h, const float* vel, int G, const int64_t* sel, int64_t nsel,
                            double* rho, double* out, double* abs_sum) {
  int64_t N = t->N, ng = sel ? nsel : (N + G - 1) / G;
  float* hs = sorted_h(t, h);
  float* bmax = (float*)malloc(4 * t->ncell); float* rsph = (float*)malloc(4 * t->ncell);
  sph_radii_sorted(t, hs, bmax, rsph);
  uint64_t total = 0;
#pragma omp parallel reduction(+ : total)
  {
    lists_t L; memset(&L, 0, sizeof L);
#pragma omp for schedule(dynamic, 1)
    for (int64_t gi = 0; gi < ng; gi++) {
      int64_t g = sel ? sel[gi] : gi;
      int64_t a = g * G, b = a + G < N ? a + G : N;
      gbox_t box = group_box(t, a, b, hs);
      L.np = 0; L.ntests = 0;
      walk_sph(t, bmax, rsph, &box, 0, &L);
      total += (uint64_t)(b - a) * (uint64_t)L.np;
      for (int64_t s = a; s < b; s++) {
        const float* pi = t->spos + 4 * s;
        int64_t io = t->perm[s];
        float hi = hs[s], h2 = hi * hi;
        double r0 = 0, dv = 0, rx = 0, ry = 0, rz = 0, as = 0;
        for (int64_t k = 0; k < L.np; k++) {
          int64_t j = L.parts[k];
          const float* pj = t->spos + 4 * j;
          if (!(r2_f32(pi, pj) < h2)) continue;
          double ex = (double)pi[0] - pj[0], ey = (double)pi[1] - pj[1], ez = (double)pi[2] - pj[2];   /* x_i - x_j */
          double r = sqrt(ex * ex + ey * ey + ez * ez);
          r0 += (double)pj[3] * orc_W(r, (double)hi);
          if (r == 0.0) continue;
          int64_t jo = t->perm[j];
          double gw = orc_dWdr(r, (double)hi) / r;                                                   /* grad_i W = gw (x_i - x_j) */
          double ux = (double)vel[4 * jo] - vel[4 * io], uy = (double)vel[4 * jo + 1] - vel[4 * io + 1],
                 uz = (double)vel[4 * jo + 2] - vel[4 * io + 2];                                     /* v_j - v_i */
          double m = pj[3];
          dv += m * gw * (ux * ex + uy * ey + uz * ez);
          /* (v_i - v_j) x grad W = -u x (gw e) = gw (e x u) */
          rx += m * gw * (ey * uz - ez * uy);
          ry += m * gw * (ez * ux - ex * uz);
          rz += m * gw * (ex * uy - ey * ux);
          as += m * fabs(gw) * r * sqrt(ux * ux + uy * uy + uz * uz);
        }
        if (rho) rho[io] = r0;
        out[4 * io] = dv / r0; out[4 * io + 1] = rx / r0; out[4 * io + 2] = ry / r0; out[4 * io + 3] = rz / r0;
        if (abs_sum) abs_sum[io] = as / r0;
      }
    }
    free(L.parts); free(L.cells);
  }
  free(hs); free(bmax); free(rsph);
  return total;
}
/* ---------------- adaptive smoothing length ("h for each particle variable", L246; BASELINE config 4
 * "adaptive to ~50 neighbours"; no rule in the paper).  Reading R21: per-particle root search on the
 * neighbour count n_i(h_i) of R16 (self included; a monotone step function of h_i alone).  Every iteration
 * counts neighbours with the current h; a particle with |n_i - n_target| <= tol is settled; otherwise its
 * bracket is updated (n_i < n_target: lo_i = h_i, else hi_i = h_i) and
 *   both ends known:  h_i <- fl32(0.5f * fl32(lo_i + hi_i))   (bisection; if that equals an end, settled)
 *   else:             h_i <- fl32( h_i * clamp(1 + (n_target - n_i) / (3 n_i), 0.7, 1.3) )   in fp64
 * (the first-order form of (n_target/n_i)^(1/3); only IEEE + - * /, so both sides get the same bits).
 * Stops when every particle is settled or after max_iter updates.  The tree is not rebuilt; radii (Eq. 5)
 * and lists are recomputed every iteration.  Returns the number of updates; nngb_out = counts of the final h. */
int orc_sph_adapt_h(const orc_tree* t, float* h, double n_target, double tol, int max_iter, int G, uint32_t* nngb_out) {
  int64_t N = t->N;
  uint32_t* n = (uint32_t*)malloc(4 * (N > 0 ? N : 1));
  double* rho = (double*)malloc(8 * (N > 0 ? N : 1));
  float* lo = (float*)calloc(N > 0 ? N : 1, 4);
  float* hi = (float*)malloc(4 * (N > 0 ? N : 1));
  unsigned char* settled = (unsigned char*)calloc(N > 0 ? N : 1, 1);
  for (int64_t i = 0; i < N; i++) hi[i] = INFINITY;
  int it = 0;
  for (;;) {
    orc_sph_density(t, h, G, rho, n, NULL, NULL);
    int64_t bad = 0;
    for (int64_t i = 0; i < N; i++) {
      if (!(fabs((double)n[i] - n_target) > tol)) settled[i] = 1;     /* also re-settles nothing: h_i is frozen once settled */
      if (!settled[i]) bad++;
    }
    if (bad == 0 || it >= max_iter) break;
    for (int64_t i = 0; i < N; i++) {
      if (settled[i]) continue;
      double ni = (double)n[i];
      if (ni < n_target) lo[i] = h[i]; else hi[i] = h[i];
      if (lo[i] > 0.0f && hi[i] < INFINITY) {
        float mid = 0.5f * (lo[i] + hi[i]);
        if (mid == lo[i] || mid == hi[i]) settled[i] = 1;             /* the step jumps over the band */
        else h[i] = mid;
      } else {
        double f = 1.0 + (n_target - ni) / (3.0 * ni);                  /* n_i >= 1: the particle itself */
        if (f < 0.7) f = 0.7;
        if (f > 1.3) f = 1.3;
        h[i] = (float)((double)h[i] * f);
      }
    }
    it++;
  }
  if (nngb_out) memcpy(nngb_out, n, 4 * N);
  free(n); free(rho); free(lo); free(hi); free(settled);
  return it;
}
void orc_sph_group_list(const orc_tree* t, const float* h, int G, int64_t g, uint32_t* part_slots) {
  float* hs = sorted_h(t, h);
  float* bmax = (float*)malloc(4 * t->ncell); float* rsph = (float*)malloc(4 * t->ncell);
  sph_radii_sorted(t, hs, bmax, rsph);
  int64_t a = g * G, b = a + G < t->N ? a + G : t->N;
  gbox_t box = group_box(t, a, b, hs);
  lists_t L; memset(&L, 0, sizeof L);
  walk_sph(t, bmax, rsph, &box, 0, &L);
  memcpy(part_slots, L.parts, 4 * L.np);
  free(L.parts); free(L.cells); free(hs); free(bmax); free(rsph);
}

/* R17: symmetric pressure force (TREESPH/GADGET form) and optional du/dt. */
/* visc != NULL (needs vel): artificial viscosity ("a hybrid of [53] and [54]", i.e. the standard
 * pair viscosity with the Balsara shear switch and a per-particle alpha; the paper prints no formula).
 * Reading R24: visc = 4N floats (c_i sound speed, alpha_i, f_i Balsara factor, -); for a pair with
 * w = (v_i - v_j).(x_i - x_j) < 0:  l = (h_i + h_j)/4,  mu = l w / (r^2 + 0.01 l^2),
 *   Pi_ij = fbar (-abar cbar mu + 2 abar mu^2) / rhobar   (bars: arithmetic means of the two particles),
 * else Pi_ij = 0; Pi_ij is added to (P_i/rho_i^2 + P_j/rho_j^2) in both the force and du/dt of R17. */
static uint64_t sph_force_impl(const orc_tree* t, const float* h, const double* rho, const double* P,
                               const float* vel, const float* visc, int G, const int64_t* sel, int64_t nsel,
                               double* out, double* abs_sum) {
  int64_t N = t->N, ng = sel ? nsel : (N + G - 1) / G;
  float* hs = sorted_h(t, h);
  float* bmax = (float*)malloc(4 * t->ncell); float* rsph = (float*)malloc(4 * t->ncell);
  sph_radii_sorted(t, hs, bmax, rsph);
  uint64_t total = 0;
#pragma omp parallel reduction(+ : total)
  {
    lists_t L; memset(&L, 0, sizeof L);
#pragma omp for schedule(dynamic, 1)
    for (int64_t gi = 0; gi < ng; gi++) {
      int64_t g = sel ? sel[gi] : gi;
      int64_t a = g * G, b = a + G < N ? a + G : N;
      gbox_t box = group_box(t, a, b, hs);
      L.np = 0; L.ntests = 0;
      walk_sph(t, bmax, rsph, &box, 0, &L);
      total += (uint64_t)(b - a) * (uint64_t)L.np;
      for (int64_t s = a; s < b; s++) {
        const float* pi = t->spos + 4 * s;
        int64_t io = t->perm[s];
        float hi = hs[s];
        double pri = P[io] / (rho[io] * rho[io]);
        double ax = 0, ay = 0, az = 0, du = 0, asum = 0, dsum = 0;
        for (int64_t k = 0; k < L.np; k++) {
          int64_t j = L.parts[k];
          if (j == s) continue;
          const float* pj = t->spos + 4 * j;
          float hj = hs[j], hm = hi > hj ? hi : hj;
          if (!(r2_f32(pi, pj) < hm * hm)) continue;   /* decision in fp32 */
          int64_t jo = t->perm[j];
          double dx = (double)pi[0] - pj[0], dy = (double)pi[1] - pj[1], dz = (double)pi[2] - pj[2];
          double r = sqrt(dx * dx + dy * dy + dz * dz);
          if (r == 0.0) continue;
          double gw = 0.5 * (orc_dWdr(r, (double)hi) + orc_dWdr(r, (double)hj)) / r;  /* grad_i W = gw * (xi-xj) */
          double Pi = 0.0;
          if (visc && vel) {
            double wx = (double)vel[4 * io] - vel[4 * jo], wy = (double)vel[4 * io + 1] - vel[4 * jo + 1],
                   wz = (double)vel[4 * io + 2] - vel[4 * jo + 2];
            double w = wx * dx + wy * dy + wz * dz;
            if (w < 0.0) {
              double l = 0.25 * ((double)hi + (double)hj);
              double mu = l * w / (r * r + 0.01 * l * l);
              double ab = 0.5 * ((double)visc[4 * io + 1] + visc[4 * jo + 1]), cb = 0.5 * ((double)visc[4 * io] + visc[4 * jo]);
              double fb = 0.5 * ((double)visc[4 * io + 2] + visc[4 * jo + 2]), rb = 0.5 * (rho[io] + rho[jo]);
              Pi = fb * (-ab * cb * mu + 2.0 * ab * mu * mu) / rb;
            }
          }
          double f = (double)pj[3] * (pri + P[jo] / (rho[jo] * rho[jo]) + Pi) * gw;
          ax -= f * dx; ay -= f * dy; az -= f * dz;
          asum += fabs(f) * r;                       /* |a_ij|, for the test's error bound */
          if (vel) {
            double vx = (double)vel[4 * io] - vel[4 * jo], vy = (double)vel[4 * io + 1] - vel[4 * jo + 1],
                   vz = (double)vel[4 * io + 2] - vel[4 * jo + 2];
            du += 0.5 * f * (vx * dx + vy * dy + vz * dz);
            dsum += fabs(0.5 * f * (vx * dx + vy * dy + vz * dz));
          }
        }
        out[4 * io] = ax; out[4 * io + 1] = ay; out[4 * io + 2] = az; out[4 * io + 3] = du;
        if (abs_sum) { abs_sum[2 * io] = asum; abs_sum[2 * io + 1] = dsum; }
      }
    }
    free(L.parts); free(L.cells);
  }
  free(hs); free(bmax); free(rsph);
  return total;
}
uint64_t orc_sph_force_sel(const orc_tree* t, const float* h, const double* rho, const double* P,
                           const float* vel, int G, const int64_t* sel, int64_t nsel, double* out, double* abs_sum) {
  return sph_force_impl(t, h, rho, P, vel, NULL, G, sel, nsel, out, abs_sum);
}
uint64_t orc_sph_force_visc_sel(const orc_tree* t, const float* h, const double* rho, const double* P,
                                const float* vel, const float* visc, int G, const int64_t* sel, int64_t nsel,
                                double* out, double* abs_sum) {
  return sph_force_impl(t, h, rho, P, vel, visc, G, sel, nsel, out, abs_sum);
}
uint64_t orc_sph_force(const orc_tree* t, const float* h, const double* rho, const double* P,
                       const float* vel, int G, double* out, double* abs_sum) {
  return orc_sph_force_sel(t, h, rho, P, vel, G, NULL, 0, out, abs_sum);
}

void orc_set_dist_kind(orc_tree* t, int kind) { t->dist_kind = kind; }
void orc_set_split_pieces(orc_tree* t, int K) { t->split_pieces = K; }
int orc_max_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}
void orc_set_threads(int n) {
#ifdef _OPENMP
  omp_set_num_threads(n);
#else
  (void)n;
#endif
}
