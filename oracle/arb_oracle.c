/* arb_oracle.c - the CPU ORACLE (see arb_oracle.h: TEST INFRASTRUCTURE, not the product).
 *
 * Plain fp64 C, one cell at a time, no blocking / fusion / layout tricks, compiled with
 * -ffp-contract=off so that every operation rounds separately.  Shares nothing with the CUDA path.
 *
 * Every function cites the passage of /root/reference/PAPER.md it follows; "Rn" are the readings
 * listed in DESIGN.md (taken from SURVEY.md 8(c)) for what the paper leaves open.
 *
 * Pins (tests/test_oracle_pins.py, all -m "not gpu"):
 *   orc_hines_solve / orc_assemble ... dense LAPACK solve on random trees (P1), symmetry and
 *                                      diagonal dominance (P2), branch-point current balance (P5)
 *   time stepping of the linear part .. closed-form cable steady state (P3) and per-step
 *                                      eigenmode decay (P4)
 *   orc_hh_rates / gate update ........ textbook constants at -65 mV, rest-potential fixed point
 *                                      (P6), removable singularities (P7), scipy solve_ivp (P9)
 *   synapse / event path .............. closed-form decay and split-step exactness (P8), step
 *                                      splitting continuity (P12), hand-computed network timings
 *                                      and the ring invariant (P11), ordering invariance (P10)
 *   synapse current I = g (V - e) ..... one-step closed form with e != 0, two synapses on one CV,
 *                                      conductance-weighted steady state (P13)
 *   "state integrated with V'" ........ hand-computed gates after one step with V' - V > 3 mV (P14)
 *   clamp window t0 <= t < t1 ......... hand-computed recurrence, exactly steps 5 and 6 see it (P15)
 * tests/test_oracle_mutations.py mutates a copy of this file line by line and checks that the pins
 * above turn red for every mutation in its list.
 * Parity unpinned (inputs / constants only, identical on both sides): HH reversal potentials and
 * temperature (R5), V_init (R4), the cell-centred generator (R3), drive and kick weights.
 *
 * Units (R2): V mV, t ms, area um^2, cm uF/cm^2, density conductance S/cm^2, point conductance uS,
 * current nA, axial resistance MOhm, capacitance nF.
 */
#include "arb_oracle.h"

#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

static char g_err[512] = "";
static int g_threads = 1;
const char* orc_last_error(void) { return g_err; }
void orc_set_threads(int n) { g_threads = n < 1 ? 1 : n; }
int orc_get_threads(void) {
#ifdef _OPENMP
  return g_threads;
#else
  return 1;
#endif
}
#define FAIL(code, ...) do { snprintf(g_err, sizeof g_err, __VA_ARGS__); return (code); } while (0)

/* ------------------------------------------------------------------------------------------
 * HH rate functions (R5: textbook Hodgkin-Huxley 1952 at 6.3 C, rest shifted to -65 mV; the paper
 * only names the mechanism).  Rates in 1/ms, V in mV.
 * ------------------------------------------------------------------------------------------ */
double orc_exprelr(double x) { return x == 0.0 ? 1.0 : x / expm1(x); }

void orc_hh_rates(double v, double out[6]) {
  out[0] = orc_exprelr(-(v + 40.0) / 10.0);           /* alpha_m = 0.1 (V+40)/(1-exp(-(V+40)/10)) */
  out[1] = 4.0 * exp(-(v + 65.0) / 18.0);             /* beta_m  */
  out[2] = 0.07 * exp(-(v + 65.0) / 20.0);            /* alpha_h */
  out[3] = 1.0 / (1.0 + exp(-(v + 35.0) / 10.0));     /* beta_h  */
  out[4] = 0.1 * orc_exprelr(-(v + 55.0) / 10.0);     /* alpha_n = 0.01 (V+55)/(1-exp(-(V+55)/10)) */
  out[5] = 0.125 * exp(-(v + 65.0) / 80.0);           /* beta_n  */
}

/* ------------------------------------------------------------------------------------------
 * PAPER.md:152-156, implicit Euler system of one cell for a step of length delta:
 *   (c_i/delta + sum_j sigma_ij) V'_i - sum_j sigma_ij V'_j = -I_i^memb + (c_i/delta) V_i .
 * Tree => one off-diagonal pair per CV i >= 1, between i and parent(i), u_i = -sigma_i.
 * C_i[nF] = cm*area*1e-5 ; sigma_i[uS] = 1/raxial_i  (R2).
 * ------------------------------------------------------------------------------------------ */
void orc_assemble(int64_t n, const int32_t* parent, const double* area, const double* cm,
                  const double* raxial, const double* v, const double* i_memb, double delta,
                  double* d, double* u, double* rhs) {
  for (int64_t i = 0; i < n; ++i) {
    double c = cm[i] * area[i] * 1e-5;
    d[i] = c / delta;
    rhs[i] = (c / delta) * v[i] - i_memb[i];
    u[i] = 0.0;
  }
  for (int64_t i = 1; i < n; ++i) {
    double sigma = 1.0 / raxial[i];
    d[i] += sigma;
    d[parent[i]] += sigma;
    u[i] = -sigma;
  }
}

/* PAPER.md:158 (Hines 1984, ref [12]): with parent < index, eliminate leaves -> root, then
 * substitute root -> leaves. */
void orc_hines_solve(int64_t n, const int32_t* parent, double* d, const double* u, double* rhs,
                     double* x) {
  for (int64_t i = n - 1; i >= 1; --i) {
    double f = u[i] / d[i];
    d[parent[i]] -= f * u[i];
    rhs[parent[i]] -= f * rhs[i];
  }
  x[0] = rhs[0] / d[0];
  for (int64_t i = 1; i < n; ++i) x[i] = (rhs[i] - u[i] * x[parent[i]]) / d[i];
}

/* ------------------------------------------------------------------------------------------ */
typedef struct { double t; int32_t syn; int64_t seq; double w; } event;

typedef struct {
  int64_t n, ns;                 /* CVs, synapses */
  int64_t cv0, syn0;             /* offsets into the model-wide arrays */
  event* q; int64_t qh, qn, qcap;/* pending events, sorted by (t, syn, seq); q[qh..qn) live */
  int64_t* clamps; int64_t n_clamps;
  int32_t det; double v_prev; int armed;
  double new_spikes[8]; int n_new;   /* spikes of the grid step in progress */
  int kind;                          /* 0 cable, 1 LIF, 2 spike source (R20) */
  double t_last, t_ref_end;          /* LIF: time V refers to; end of the refractory period */
  int64_t src_cur;                   /* source: next scheduled spike */
  int spike_overflow;                /* a ninth spike in one grid step: orc_advance reports it, nothing is dropped silently */
  int64_t substeps;
} cell_t;

struct orc_model {
  int64_t n_cells, n_cv, n_syn, n_clamp, n_conn;
  /* copies of the description */
  int32_t* parent; double *area, *cm, *rax, *gna, *gk, *gl, *pg, *pe;
  double ena, ek, el, theta;
  double *lif_tau_m, *lif_v_th, *lif_c_m, *lif_e_l, *lif_e_r, *lif_t_ref;
  int64_t* src_off; double* src_time;
  int32_t* syn_cv; double *syn_tau, *syn_e;
  double *cl_t0, *cl_t1, *cl_amp; int32_t* cl_cv;
  int64_t *out_off, *out_k;      /* connections grouped by source, ascending k inside a group */
  int64_t* conn_dst; int32_t* conn_syn; double *conn_delay, *conn_w;
  double min_delay;
  /* state */
  double *v, *m, *h, *nn, *g;
  double *scr;                   /* 5*n_cv scratch: I, d, u, rhs, x */
  cell_t* cells;
  double t; int64_t seq, grid_steps;
  int linearised;                /* 0: explicit membrane currents (R1); 1: conductance-linearised step (NEXT-2) */
  int64_t* sp_cell; double* sp_time; int64_t n_sp, sp_cap;
};

static int ev_less(const event* a, const event* b) {
  if (a->t != b->t) return a->t < b->t;
  if (a->syn != b->syn) return a->syn < b->syn;
  return a->seq < b->seq;
}

static int ev_cmp(const void* a, const void* b) {
  return ev_less((const event*)a, (const event*)b) ? -1 : (ev_less((const event*)b, (const event*)a) ? 1 : 0);
}

static int q_reserve(cell_t* c) {
  if (c->qn < c->qcap) return 0;
  if (c->qh > 0) {              /* drop delivered prefix */
    memmove(c->q, c->q + c->qh, (size_t)(c->qn - c->qh) * sizeof(event));
    c->qn -= c->qh; c->qh = 0;
    if (c->qn < c->qcap) return 0;
  }
  int64_t cap = c->qcap ? 2 * c->qcap : 16;
  event* nq = (event*)realloc(c->q, (size_t)cap * sizeof(event));
  if (!nq) return -1;
  c->q = nq; c->qcap = cap;
  return 0;
}

/* keep the queue ordered by (time, synapse, insertion order) - R9 */
static int q_insert(cell_t* c, event e) {
  if (q_reserve(c)) return -1;
  int64_t lo = c->qh, hi = c->qn;
  while (lo < hi) { int64_t mid = (lo + hi) / 2; if (ev_less(&e, &c->q[mid])) hi = mid; else lo = mid + 1; }
  memmove(c->q + lo + 1, c->q + lo, (size_t)(c->qn - lo) * sizeof(event));
  c->q[lo] = e; c->qn++;
  return 0;
}

static int has_hh(const orc_model* M, int64_t i) {
  return M->gna && (M->gna[i] != 0.0 || M->gk[i] != 0.0 || M->gl[i] != 0.0);
}

/* Step 2 of SURVEY.md 8(c) / PAPER.md:148 "at a time t, the synapse, channel and injection
 * currents are calculated as a function of V_i(t)"; terms of PAPER.md:127-131 (eq 2a), nA. */
static void cell_currents(const orc_model* M, const cell_t* c, double t, double* I) {
  const double* v = M->v + c->cv0;
  for (int64_t i = 0; i < c->n; ++i) {
    int64_t gi = c->cv0 + i;
    I[i] = 0.0;
    if (has_hh(M, gi)) {
      double m = M->m[gi], h = M->h[gi], n = M->nn[gi];
      double dens = M->gna[gi] * m * m * m * h * (v[i] - M->ena) + M->gk[gi] * n * n * n * n * (v[i] - M->ek) +
                    M->gl[gi] * (v[i] - M->el);             /* mA/cm^2 */
      I[i] += dens * M->area[gi] * 1e-2;
    }
    if (M->pg && M->pg[gi] != 0.0) I[i] += M->pg[gi] * (v[i] - M->pe[gi]) * M->area[gi] * 1e-2;
  }
  for (int64_t s = 0; s < c->ns; ++s) {                      /* ascending synapse index */
    int64_t gs = c->syn0 + s; int32_t i = M->syn_cv[gs];
    I[i] += M->g[gs] * (v[i] - M->syn_e[gs]);                /* R7: uS * mV = nA */
  }
  for (int64_t k = 0; k < c->n_clamps; ++k) {                /* R8: positive amplitude depolarises */
    int64_t ck = c->clamps[k];
    if (M->cl_t0[ck] <= t && t < M->cl_t1[ck]) I[M->cl_cv[ck]] -= M->cl_amp[ck];
  }
}

/* SURVEY.md 8(f) NEXT-2, the conductance-linearised variant of the implicit Euler equation at PAPER.md:152-156:
 * every membrane current of the form g_k (V - E_k) is taken at the NEW voltage,
 *   (c_i/delta + sum_j sigma_ij + sum_k g_k) V'_i - sum_j sigma_ij V'_j = (c_i/delta) V_i + sum_k g_k E_k + I_i^inj ,
 * with the conductances g_k from the state at time t (HH: gnabar m^3 h, gkbar n^4, gl; passive g; synapses g_s),
 * so the matrix is assembled and eliminated afresh every step.  gsum_i = sum_k g_k [uS], src_i = sum_k g_k E_k
 * + clamp currents [nA]. */
static void cell_conductances(const orc_model* M, const cell_t* c, double t, double* gsum, double* src) {
  for (int64_t i = 0; i < c->n; ++i) {
    int64_t gi = c->cv0 + i;
    gsum[i] = 0.0; src[i] = 0.0;
    if (has_hh(M, gi)) {
      double m = M->m[gi], h = M->h[gi], n = M->nn[gi], sc = M->area[gi] * 1e-2;
      double gna = M->gna[gi] * m * m * m * h * sc, gk = M->gk[gi] * n * n * n * n * sc, gl = M->gl[gi] * sc;
      gsum[i] += gna + gk + gl;
      src[i] += gna * M->ena + gk * M->ek + gl * M->el;
    }
    if (M->pg && M->pg[gi] != 0.0) {
      double g = M->pg[gi] * M->area[gi] * 1e-2;
      gsum[i] += g;
      src[i] += g * M->pe[gi];
    }
  }
  for (int64_t s = 0; s < c->ns; ++s) {                      /* ascending synapse index */
    int64_t gs = c->syn0 + s; int32_t i = M->syn_cv[gs];
    gsum[i] += M->g[gs];
    src[i] += M->g[gs] * M->syn_e[gs];
  }
  for (int64_t k = 0; k < c->n_clamps; ++k) {                /* R8: a current source, not a conductance */
    int64_t ck = c->clamps[k];
    if (M->cl_t0[ck] <= t && t < M->cl_t1[ck]) src[M->cl_cv[ck]] += M->cl_amp[ck];
  }
}

/* One (sub-)step of one cell from t to t+delta: steps 2-7 of SURVEY.md 8(c). */
static void cell_step(orc_model* M, cell_t* c, double t, double delta) {
  double* I = M->scr + 5 * c->cv0;
  double *d = I + c->n, *u = d + c->n, *rhs = u + c->n, *x = rhs + c->n;
  double* v = M->v + c->cv0;
  if (!M->linearised) {
    cell_currents(M, c, t, I);
    orc_assemble(c->n, M->parent + c->cv0, M->area + c->cv0, M->cm + c->cv0, M->rax + c->cv0, v, I, delta, d, u, rhs);
  } else {
    /* assemble with no current (I = 0), then the conductances go on the diagonal and their sources on the rhs;
     * x serves as scratch for src until the solve overwrites it */
    for (int64_t i = 0; i < c->n; ++i) I[i] = 0.0;
    orc_assemble(c->n, M->parent + c->cv0, M->area + c->cv0, M->cm + c->cv0, M->rax + c->cv0, v, I, delta, d, u, rhs);
    cell_conductances(M, c, t, I, x);
    for (int64_t i = 0; i < c->n; ++i) { d[i] += I[i]; rhs[i] += x[i]; }
  }
  orc_hines_solve(c->n, M->parent + c->cv0, d, u, rhs, x);
  c->v_prev = v[c->det];
  for (int64_t i = 0; i < c->n; ++i) v[i] = x[i];            /* V <- V' */
  /* PAPER.md:148 "finally, the state variables are integrated with the updated voltage values";
   * R5: exact exponential for frozen V', R7: g <- g exp(-delta/tau). */
  for (int64_t i = 0; i < c->n; ++i) {
    int64_t gi = c->cv0 + i;
    if (!has_hh(M, gi)) continue;
    double r[6];
    orc_hh_rates(v[i], r);
    double* st[3] = { &M->m[gi], &M->h[gi], &M->nn[gi] };
    for (int k = 0; k < 3; ++k) {
      double a = r[2 * k], b = r[2 * k + 1];
      double xinf = a / (a + b);
      *st[k] = xinf + (*st[k] - xinf) * exp(-delta * (a + b));
    }
  }
  for (int64_t s = 0; s < c->ns; ++s) {
    int64_t gs = c->syn0 + s;
    M->g[gs] = M->g[gs] * exp(-delta / M->syn_tau[gs]);
  }
  /* PAPER.md:98 threshold detector, R10: upward crossing, linear interpolation, re-arm below. */
  double vd = v[c->det];
  if (c->armed && c->v_prev < M->theta && M->theta <= vd) {
    if (c->n_new < 8) c->new_spikes[c->n_new++] = t + delta * (M->theta - c->v_prev) / (vd - c->v_prev);
    else c->spike_overflow = 1;
    c->armed = 0;
  }
  if (vd < M->theta) c->armed = 1;
  c->substeps++;
}

/* One grid interval [ta, tb] of one cell, split at event times (R9). */
static void cell_interval(orc_model* M, cell_t* c, double ta, double tb, double dt, int nominal) {
  double t = ta;
  for (;;) {
    while (c->qh < c->qn && c->q[c->qh].t <= t) {             /* deliver: g += w */
      M->g[c->syn0 + c->q[c->qh].syn] += c->q[c->qh].w;
      c->qh++;
    }
    double next = tb;
    if (c->qh < c->qn && c->q[c->qh].t < tb) next = c->q[c->qh].t;
    double delta = (nominal && t == ta && next == tb) ? dt : next - t;
    cell_step(M, c, t, delta);
    t = next;                                                 /* assigned, never accumulated */
    if (t == tb) break;
  }
}

/* Leaky integrate-and-fire cell (PAPER.md:170 names the kind only; reading R20): between events the membrane
 * potential relaxes exactly, V(t) = E_L + (V(t_last) - E_L) exp(-(t - t_last)/tau_m); an event of weight w (a charge,
 * pC = nA ms; C_m in nF) adds w / C_m [mV] to V; V >= V_th at an event emits a spike AT the event time,
 * V <- E_R, and events are ignored for t_ref, after which relaxation resumes from E_R.  Event-driven and exact: the
 * time grid plays no role.  Events with time < tb are processed in the grid interval that ends at tb. */
static void lif_interval(orc_model* M, cell_t* c, int64_t ci, double tb) {
  double* v = M->v + c->cv0;
  while (c->qh < c->qn && c->q[c->qh].t < tb) {
    const double te = c->q[c->qh].t, w = c->q[c->qh].w;
    c->qh++;
    if (te < c->t_ref_end) continue;                          /* refractory: the event is lost */
    v[0] = M->lif_e_l[ci] + (v[0] - M->lif_e_l[ci]) * exp(-(te - c->t_last) / M->lif_tau_m[ci]);
    c->t_last = te;
    v[0] += w / M->lif_c_m[ci];
    if (v[0] >= M->lif_v_th[ci]) {
      if (c->n_new < 8) c->new_spikes[c->n_new++] = te; else c->spike_overflow = 1;
      v[0] = M->lif_e_r[ci];
      c->t_ref_end = te + M->lif_t_ref[ci];
      c->t_last = c->t_ref_end;
    }
  }
}

/* Spike source ("artificial spike sources"; R20): emits its schedule, times in [ta, tb). */
static void source_interval(orc_model* M, cell_t* c, int64_t ci, double tb) {
  while (c->src_cur < M->src_off[ci + 1] && M->src_time[c->src_cur] < tb) {
    if (c->n_new < 8) c->new_spikes[c->n_new++] = M->src_time[c->src_cur]; else c->spike_overflow = 1;
    c->src_cur++;
  }
}

/* ------------------------------------------------------------------------------------------ */
static void* dup_arr(const void* p, size_t bytes) {
  if (!p) return NULL;
  void* q = malloc(bytes ? bytes : 1);
  if (q && bytes) memcpy(q, p, bytes);
  return q;
}

static int bad(double x) { return !(x == x) || x > 1.7e308 || x < -1.7e308; }

int orc_create(const orc_desc* D, orc_model** out) {
  if (!D || !out) FAIL(-1, "null argument");
  if (D->n_cells < 0 || (D->n_cells > 0 && (!D->cv_off || !D->cv_parent || !D->cv_area || !D->cv_cm || !D->cv_raxial)))
    FAIL(-1, "null compartment arrays");
  int64_t nc = D->n_cells, ncv = nc ? D->cv_off[nc] : 0, nsyn = (nc && D->syn_off) ? D->syn_off[nc] : 0;
  if ((D->hh_gnabar != NULL) != (D->hh_gkbar != NULL) || (D->hh_gnabar != NULL) != (D->hh_gl != NULL))
    FAIL(-2, "hh arrays must be all given or all NULL");
  if ((D->pas_g != NULL) != (D->pas_e != NULL)) FAIL(-2, "pas arrays must be both given or both NULL");
  for (int64_t c = 0; c < nc; ++c) {
    int64_t n = D->cv_off[c + 1] - D->cv_off[c];
    if (n < 1) FAIL(-2, "cell %lld has no compartments", (long long)c);
    for (int64_t i = 0; i < n; ++i) {
      int64_t gi = D->cv_off[c] + i; int32_t p = D->cv_parent[gi];
      if ((i == 0 && p != -1) || (i > 0 && (p < 0 || p >= i))) FAIL(-2, "cell %lld cv %lld: bad parent %d", (long long)c, (long long)i, p);
      if (!(D->cv_area[gi] > 0) || !(D->cv_cm[gi] > 0) || bad(D->cv_area[gi]) || bad(D->cv_cm[gi])) FAIL(-2, "non-positive area/cm");
      if (i > 0 && (!(D->cv_raxial[gi] > 0) || bad(D->cv_raxial[gi]))) FAIL(-2, "non-positive axial resistance");
      if (D->cv_vinit && bad(D->cv_vinit[gi])) FAIL(-2, "non-finite vinit");
      if (D->hh_gnabar && (bad(D->hh_gnabar[gi]) || bad(D->hh_gkbar[gi]) || bad(D->hh_gl[gi]))) FAIL(-2, "non-finite hh parameter");
      if (D->pas_g && (bad(D->pas_g[gi]) || bad(D->pas_e[gi]))) FAIL(-2, "non-finite pas parameter");
    }
    int64_t s0 = D->syn_off ? D->syn_off[c] : 0, s1 = D->syn_off ? D->syn_off[c + 1] : 0;
    if (s1 < s0) FAIL(-2, "syn_off not monotone");
    for (int64_t s = s0; s < s1; ++s) {
      if (D->syn_cv[s] < 0 || D->syn_cv[s] >= n) FAIL(-2, "synapse cv out of range");
      if (!(D->syn_tau[s] > 0) || bad(D->syn_tau[s]) || bad(D->syn_e[s])) FAIL(-2, "bad synapse parameter");
    }
    if (D->det_cv && (D->det_cv[c] < 0 || D->det_cv[c] >= n)) FAIL(-2, "detector cv out of range");
  }
  if (bad(D->threshold) || bad(D->hh_ena) || bad(D->hh_ek) || bad(D->hh_el)) FAIL(-2, "non-finite scalar");
  for (int64_t k = 0; k < D->n_clamp; ++k) {
    int64_t c = D->clamp_cell[k];
    if (c < 0 || c >= nc || D->clamp_cv[k] < 0 || D->clamp_cv[k] >= D->cv_off[c + 1] - D->cv_off[c]) FAIL(-2, "clamp out of range");
    if (D->clamp_t0[k] != D->clamp_t0[k] || D->clamp_t1[k] != D->clamp_t1[k] || bad(D->clamp_amp[k])) FAIL(-2, "bad clamp");
  }
  double min_delay = INFINITY;
  for (int64_t k = 0; k < D->n_conn; ++k) {
    int64_t s = D->conn_src[k], d = D->conn_dst[k];
    if (s < 0 || s >= nc || d < 0 || d >= nc) FAIL(-2, "connection cell out of range");
    if (D->conn_syn[k] < 0 || D->conn_syn[k] >= D->syn_off[d + 1] - D->syn_off[d]) FAIL(-2, "connection synapse out of range");
    if (!(D->conn_delay[k] > 0) || bad(D->conn_delay[k]) || bad(D->conn_weight[k])) FAIL(-2, "connection delay must be > 0");
    if (D->conn_delay[k] < min_delay) min_delay = D->conn_delay[k];
  }
  for (int64_t k = 0; k < D->n_ext; ++k) {
    int64_t c = D->ext_cell[k];
    if (c < 0 || c >= nc) FAIL(-2, "external event cell out of range");
    if (D->ext_syn[k] < 0 || D->ext_syn[k] >= D->syn_off[c + 1] - D->syn_off[c]) FAIL(-2, "external event synapse out of range");
    if (!(D->ext_time[k] >= 0) || bad(D->ext_time[k]) || bad(D->ext_weight[k])) FAIL(-2, "external event earlier than t=0 or non-finite");
  }

  orc_model* M = (orc_model*)calloc(1, sizeof *M);
  if (!M) FAIL(-5, "out of memory");
  M->n_cells = nc; M->n_cv = ncv; M->n_syn = nsyn; M->n_clamp = D->n_clamp; M->n_conn = D->n_conn;
  M->min_delay = min_delay;
  M->parent = (int32_t*)dup_arr(D->cv_parent, (size_t)ncv * 4);
  M->area = (double*)dup_arr(D->cv_area, (size_t)ncv * 8);
  M->cm = (double*)dup_arr(D->cv_cm, (size_t)ncv * 8);
  M->rax = (double*)dup_arr(D->cv_raxial, (size_t)ncv * 8);
  M->gna = (double*)dup_arr(D->hh_gnabar, (size_t)ncv * 8);
  M->gk = (double*)dup_arr(D->hh_gkbar, (size_t)ncv * 8);
  M->gl = (double*)dup_arr(D->hh_gl, (size_t)ncv * 8);
  M->pg = (double*)dup_arr(D->pas_g, (size_t)ncv * 8);
  M->pe = (double*)dup_arr(D->pas_e, (size_t)ncv * 8);
  M->ena = D->hh_ena; M->ek = D->hh_ek; M->el = D->hh_el; M->theta = D->threshold;
  M->syn_cv = (int32_t*)dup_arr(D->syn_cv, (size_t)nsyn * 4);
  M->syn_tau = (double*)dup_arr(D->syn_tau, (size_t)nsyn * 8);
  M->syn_e = (double*)dup_arr(D->syn_e, (size_t)nsyn * 8);
  M->cl_cv = (int32_t*)dup_arr(D->clamp_cv, (size_t)D->n_clamp * 4);
  M->cl_t0 = (double*)dup_arr(D->clamp_t0, (size_t)D->n_clamp * 8);
  M->cl_t1 = (double*)dup_arr(D->clamp_t1, (size_t)D->n_clamp * 8);
  M->cl_amp = (double*)dup_arr(D->clamp_amp, (size_t)D->n_clamp * 8);
  M->conn_dst = (int64_t*)dup_arr(D->conn_dst, (size_t)D->n_conn * 8);
  M->conn_syn = (int32_t*)dup_arr(D->conn_syn, (size_t)D->n_conn * 4);
  M->conn_delay = (double*)dup_arr(D->conn_delay, (size_t)D->n_conn * 8);
  M->conn_w = (double*)dup_arr(D->conn_weight, (size_t)D->n_conn * 8);
  if (D->cell_kind) {
    M->lif_tau_m = (double*)dup_arr(D->lif_tau_m, (size_t)nc * 8); M->lif_v_th = (double*)dup_arr(D->lif_v_th, (size_t)nc * 8);
    M->lif_c_m = (double*)dup_arr(D->lif_c_m, (size_t)nc * 8); M->lif_e_l = (double*)dup_arr(D->lif_e_l, (size_t)nc * 8);
    M->lif_e_r = (double*)dup_arr(D->lif_e_r, (size_t)nc * 8); M->lif_t_ref = (double*)dup_arr(D->lif_t_ref, (size_t)nc * 8);
    if (D->src_off) {
      M->src_off = (int64_t*)dup_arr(D->src_off, (size_t)(nc + 1) * 8);
      M->src_time = (double*)dup_arr(D->src_time, (size_t)D->src_off[nc] * 8);
    }
  }
  M->v = (double*)calloc((size_t)ncv + 1, 8); M->m = (double*)calloc((size_t)ncv + 1, 8);
  M->h = (double*)calloc((size_t)ncv + 1, 8); M->nn = (double*)calloc((size_t)ncv + 1, 8);
  M->g = (double*)calloc((size_t)nsyn + 1, 8);
  M->scr = (double*)calloc(5 * (size_t)ncv + 1, 8);
  M->cells = (cell_t*)calloc((size_t)nc + 1, sizeof(cell_t));
  M->out_off = (int64_t*)calloc((size_t)nc + 2, 8);
  M->out_k = (int64_t*)calloc((size_t)D->n_conn + 1, 8);

  /* R4: V = vinit or -65 mV, gates at their steady state for that V, g = 0, t = 0. */
  for (int64_t i = 0; i < ncv; ++i) {
    M->v[i] = D->cv_vinit ? D->cv_vinit[i] : -65.0;
    if (has_hh(M, i)) {
      double r[6]; orc_hh_rates(M->v[i], r);
      M->m[i] = r[0] / (r[0] + r[1]); M->h[i] = r[2] / (r[2] + r[3]); M->nn[i] = r[4] / (r[4] + r[5]);
    }
  }
  /* connections grouped by source cell, ascending k within a source (R13) */
  for (int64_t k = 0; k < D->n_conn; ++k) M->out_off[D->conn_src[k] + 1]++;
  for (int64_t c = 0; c < nc; ++c) M->out_off[c + 1] += M->out_off[c];
  { int64_t* cur = (int64_t*)dup_arr(M->out_off, (size_t)(nc + 1) * 8);
    for (int64_t k = 0; k < D->n_conn; ++k) M->out_k[cur[D->conn_src[k]]++] = k;
    free(cur); }
  int64_t* ncl = (int64_t*)calloc((size_t)nc + 1, 8);
  for (int64_t k = 0; k < D->n_clamp; ++k) ncl[D->clamp_cell[k]]++;
  for (int64_t c = 0; c < nc; ++c) {
    cell_t* ce = &M->cells[c];
    ce->cv0 = D->cv_off[c]; ce->n = D->cv_off[c + 1] - D->cv_off[c];
    ce->syn0 = D->syn_off ? D->syn_off[c] : 0; ce->ns = D->syn_off ? D->syn_off[c + 1] - D->syn_off[c] : 0;
    ce->det = D->det_cv ? D->det_cv[c] : 0;
    ce->armed = 1; ce->v_prev = M->v[ce->cv0 + ce->det];
    ce->kind = D->cell_kind ? D->cell_kind[c] : 0;
    ce->t_last = 0.0; ce->t_ref_end = -INFINITY;
    ce->src_cur = (ce->kind == 2 && M->src_off) ? M->src_off[c] : 0;
    if (ce->kind == 1 && (!D->lif_tau_m || !(D->lif_tau_m[c] > 0) || !(D->lif_c_m[c] > 0) || !(D->lif_t_ref[c] >= 0))) {
      orc_destroy(M); FAIL(-2, "bad LIF parameters"); }
    if (ce->kind != 0 && ce->n != 1) { orc_destroy(M); FAIL(-2, "a LIF / source cell owns exactly one control volume"); }
    if (ce->kind == 2 && !M->src_off) { orc_destroy(M); FAIL(-2, "spike sources need a schedule"); }
    ce->clamps = (int64_t*)calloc((size_t)ncl[c] + 1, 8);
  }
  for (int64_t k = 0; k < D->n_clamp; ++k) { cell_t* ce = &M->cells[D->clamp_cell[k]]; ce->clamps[ce->n_clamps++] = k; }
  free(ncl);
  /* external events go straight into the queues (R14); bulk append then sort once */
  for (int64_t k = 0; k < D->n_ext; ++k) {
    cell_t* ce = &M->cells[D->ext_cell[k]];
    if (q_reserve(ce)) { orc_destroy(M); FAIL(-5, "out of memory"); }
    event e = { D->ext_time[k], D->ext_syn[k], M->seq++, D->ext_weight[k] };
    ce->q[ce->qn++] = e;
  }
  for (int64_t c = 0; c < nc; ++c) if (M->cells[c].qn > 1) qsort(M->cells[c].q, (size_t)M->cells[c].qn, sizeof(event), ev_cmp);
  *out = M;
  return 0;
}

static int push_spike(orc_model* M, int64_t cell, double t) {
  if (M->n_sp == M->sp_cap) {
    int64_t cap = M->sp_cap ? 2 * M->sp_cap : 1024;
    int64_t* a = (int64_t*)realloc(M->sp_cell, (size_t)cap * 8);
    if (!a) return -1;
    M->sp_cell = a;
    double* b = (double*)realloc(M->sp_time, (size_t)cap * 8);
    if (!b) return -1;
    M->sp_time = b; M->sp_cap = cap;
  }
  M->sp_cell[M->n_sp] = cell; M->sp_time[M->n_sp] = t; M->n_sp++;
  return 0;
}

/* Global loop of SURVEY.md 8(c): grid t_k = t0 + k*dt (by multiplication; the last point is
 * t_end itself), every cell integrates interval k, then the spikes of that interval become events
 * ((source, destination, synapse, delay, weight); event time = spike + delay).
 * The paper's epochs of Delta_T/2 are scheduling, not semantics (R12). */
int orc_advance(orc_model* M, double t_end, double dt) {
  if (!M) FAIL(-1, "null model");
  if (!(dt > 0) || bad(dt) || bad(t_end)) FAIL(-2, "dt must be > 0 and finite");
  if (t_end < M->t) FAIL(-2, "t_end earlier than current time");
  if (M->n_conn > 0 && M->min_delay < dt) FAIL(-2, "connection delay shorter than dt");
  if (t_end == M->t) return 0;
  double t0 = M->t;
  int64_t nsteps = (int64_t)ceil((t_end - t0) / dt - 1e-9);
  if (nsteps < 1) nsteps = 1;
  int last_full = fabs((t0 + (double)nsteps * dt) - t_end) <= 1e-9 * dt;
  for (int64_t k = 0; k < nsteps; ++k) {
    double ta = (k == 0) ? t0 : t0 + (double)k * dt;
    double tb = (k + 1 == nsteps) ? t_end : t0 + (double)(k + 1) * dt;
    int nominal = (k + 1 < nsteps) || last_full;
#ifdef _OPENMP
#pragma omp parallel for schedule(dynamic, 16) num_threads(g_threads)
#endif
    for (int64_t c = 0; c < M->n_cells; ++c) {
      M->cells[c].n_new = 0;
      if (M->cells[c].kind == 0) cell_interval(M, &M->cells[c], ta, tb, dt, nominal);
      else if (M->cells[c].kind == 1) lif_interval(M, &M->cells[c], c, tb);
      else source_interval(M, &M->cells[c], c, tb);
    }
    for (int64_t c = 0; c < M->n_cells; ++c)
      if (M->cells[c].spike_overflow) FAIL(-6, "cell %lld fired more than 8 spikes in one grid step", (long long)c);
    for (int64_t c = 0; c < M->n_cells; ++c) {
      cell_t* ce = &M->cells[c];
      for (int j = 0; j < ce->n_new; ++j) {
        double ts = ce->new_spikes[j];
        if (push_spike(M, c, ts)) FAIL(-5, "out of memory");
        for (int64_t o = M->out_off[c]; o < M->out_off[c + 1]; ++o) {
          int64_t kk = M->out_k[o];
          event e = { ts + M->conn_delay[kk], M->conn_syn[kk], M->seq++, M->conn_w[kk] };
          if (q_insert(&M->cells[M->conn_dst[kk]], e)) FAIL(-5, "out of memory");
        }
      }
    }
    M->grid_steps++;
  }
  M->t = t_end;
  return 0;
}

typedef struct { double t; int64_t c; } spk;
static int spk_cmp(const void* a, const void* b) {
  const spk *x = (const spk*)a, *y = (const spk*)b;
  if (x->t != y->t) return x->t < y->t ? -1 : 1;
  return x->c < y->c ? -1 : (x->c > y->c ? 1 : 0);
}

int64_t orc_spikes(orc_model* M, int64_t* cell, double* time, int64_t cap) {
  if (!M) return -1;
  if (cap > 0 && cell && time && M->n_sp > 0) {
    spk* s = (spk*)malloc((size_t)M->n_sp * sizeof(spk));
    if (!s) return -5;
    for (int64_t i = 0; i < M->n_sp; ++i) { s[i].t = M->sp_time[i]; s[i].c = M->sp_cell[i]; }
    qsort(s, (size_t)M->n_sp, sizeof(spk), spk_cmp);
    for (int64_t i = 0; i < M->n_sp && i < cap; ++i) { cell[i] = s[i].c; time[i] = s[i].t; }
    free(s);
  }
  return M->n_sp;
}

int orc_voltage(orc_model* M, double* out, int64_t n_cv) {
  if (!M || !out) FAIL(-1, "null argument");
  if (n_cv != M->n_cv) FAIL(-2, "n_cv mismatch");
  memcpy(out, M->v, (size_t)n_cv * 8);
  for (int64_t c = 0; c < M->n_cells; ++c) {                  /* LIF: the potential relaxed to the current time */
    const cell_t* ce = &M->cells[c];
    if (ce->kind == 1 && M->t > ce->t_last)
      out[ce->cv0] = M->lif_e_l[c] + (M->v[ce->cv0] - M->lif_e_l[c]) * exp(-(M->t - ce->t_last) / M->lif_tau_m[c]);
  }
  return 0;
}

int orc_probe(orc_model* M, int what, double* out, int64_t n) {
  if (!M || !out) FAIL(-1, "null argument");
  switch (what) {
    case ORC_PROBE_M: case ORC_PROBE_H: case ORC_PROBE_N: {
      if (n != M->n_cv) FAIL(-2, "size mismatch");
      const double* src = what == ORC_PROBE_M ? M->m : (what == ORC_PROBE_H ? M->h : M->nn);
      for (int64_t i = 0; i < n; ++i) out[i] = has_hh(M, i) ? src[i] : 0.0;
      return 0; }
    case ORC_PROBE_SYN_G:
      if (n != M->n_syn) FAIL(-2, "size mismatch");
      memcpy(out, M->g, (size_t)n * 8); return 0;
    case ORC_PROBE_TIME:
      if (n < 1) FAIL(-2, "size mismatch");
      out[0] = M->t; return 0;
    case ORC_PROBE_NSTEPS: {
      if (n < 2) FAIL(-2, "size mismatch");
      int64_t s = 0; for (int64_t c = 0; c < M->n_cells; ++c) s += M->cells[c].substeps;
      out[0] = (double)M->grid_steps; out[1] = (double)s; return 0; }
  }
  FAIL(-2, "unknown probe");
}

int orc_cell_currents(orc_model* M, int64_t cell, double* i_out) {
  if (!M || !i_out) FAIL(-1, "null argument");
  if (cell < 0 || cell >= M->n_cells) FAIL(-2, "cell out of range");
  cell_currents(M, &M->cells[cell], M->t, i_out);
  return 0;
}

int orc_set_state(orc_model* M, const double* v, const double* hm, const double* hh, const double* hn, const double* syn_g) {
  if (!M) FAIL(-1, "null model");
  if (v) memcpy(M->v, v, (size_t)M->n_cv * 8);
  if (hm) memcpy(M->m, hm, (size_t)M->n_cv * 8);
  if (hh) memcpy(M->h, hh, (size_t)M->n_cv * 8);
  if (hn) memcpy(M->nn, hn, (size_t)M->n_cv * 8);
  if (syn_g) memcpy(M->g, syn_g, (size_t)M->n_syn * 8);
  for (int64_t c = 0; c < M->n_cells; ++c) {
    M->cells[c].v_prev = M->v[M->cells[c].cv0 + M->cells[c].det]; M->cells[c].armed = 1;
    if (v && M->cells[c].kind == 1) { M->cells[c].t_last = M->t; M->cells[c].t_ref_end = -INFINITY; }   /* V given at the current time */
  }
  return 0;
}

int orc_set_linearised(orc_model* M, int on) {
  if (!M) FAIL(-1, "null model");
  M->linearised = on != 0;
  return 0;
}

void orc_destroy(orc_model* M) {
  if (!M) return;
  for (int64_t c = 0; c < M->n_cells; ++c) { free(M->cells[c].q); free(M->cells[c].clamps); }
  free(M->parent); free(M->area); free(M->cm); free(M->rax); free(M->gna); free(M->gk); free(M->gl);
  free(M->pg); free(M->pe); free(M->syn_cv); free(M->syn_tau); free(M->syn_e); free(M->cl_cv);
  free(M->cl_t0); free(M->cl_t1); free(M->cl_amp); free(M->conn_dst); free(M->conn_syn);
  free(M->conn_delay); free(M->conn_w); free(M->v); free(M->m); free(M->h); free(M->nn); free(M->g);
  free(M->lif_tau_m); free(M->lif_v_th); free(M->lif_c_m); free(M->lif_e_l); free(M->lif_e_r); free(M->lif_t_ref);
  free(M->src_off); free(M->src_time);
  free(M->scr); free(M->cells); free(M->out_off); free(M->out_k); free(M->sp_cell); free(M->sp_time);
  free(M);
}
