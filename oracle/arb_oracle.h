/* arb_oracle.h - C interface of the CPU ORACLE.
 *
 * TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / `--impl reference` legs may use anything under oracle/.  The CUDA library under
 * paper_1901_07454_b200/ shares no code, header, table or helper with this directory.
 *
 * What it is: a plain, slow, fp64, one-cell-at-a-time implementation of the per-time-step
 * integration of multi-compartment cells described in PAPER.md section II (lines 92-158), written
 * step by step in the paper's order with the readings R1-R17 listed in
 * DESIGN.md for everything the paper leaves open.
 */
#ifndef ARB_ORACLE_H
#define ARB_ORACLE_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

/* Problem statement (same content as the product's arb_desc, declared independently):
 * cells = trees of control volumes, mechanisms, connections as
 * (source, destination, synapse, delay, weight), threshold detectors. */
typedef struct {
  int64_t n_cells;
  const int64_t* cv_off;      /* [n_cells+1] */
  const int32_t* cv_parent;   /* [n_cv] cell-local parent, -1 for CV 0, parent < index */
  const double* cv_area;      /* um^2 */
  const double* cv_cm;        /* uF/cm^2 */
  const double* cv_raxial;    /* MOhm, centre -> parent centre */
  const double* cv_vinit;     /* mV or NULL => -65 */
  const double *hh_gnabar, *hh_gkbar, *hh_gl; /* S/cm^2 per CV, or NULL */
  double hh_ena, hh_ek, hh_el;                /* mV */
  const double *pas_g, *pas_e;                /* S/cm^2, mV, or NULL */
  const int64_t* syn_off;     /* [n_cells+1] */
  const int32_t* syn_cv;      /* cell-local CV of each synapse */
  const double *syn_tau, *syn_e;
  int64_t n_clamp;
  const int64_t* clamp_cell;
  const int32_t* clamp_cv;
  const double *clamp_t0, *clamp_t1, *clamp_amp;
  const int32_t* det_cv;      /* [n_cells] or NULL => CV 0 */
  double threshold;
  int64_t n_conn;
  const int64_t *conn_src, *conn_dst;
  const int32_t* conn_syn;    /* synapse index local to the destination cell */
  const double *conn_delay, *conn_weight;
  int64_t n_ext;
  const int64_t* ext_cell;
  const int32_t* ext_syn;
  const double *ext_time, *ext_weight;
  /* cell kinds other than the multi-compartment cell (reading R20):
   * cell_kind[c] = 0 cable cell, 1 leaky integrate-and-fire cell, 2 spike source; NULL => all cable.
   * A LIF / source cell still owns ONE control volume in the per-CV arrays (its area etc. are ignored; the CV's
   * voltage is the LIF membrane potential, vinit its initial value) and its synapse range is its event targets. */
  const int32_t* cell_kind;
  const double *lif_tau_m, *lif_v_th, *lif_c_m, *lif_e_l, *lif_e_r, *lif_t_ref;   /* [n_cells]: ms, mV, nF, mV, mV, ms */
  const int64_t* src_off;     /* [n_cells+1] spike schedule of every cell (empty unless it is a source) */
  const double* src_time;     /* ascending inside a cell */
} orc_desc;

typedef struct orc_model orc_model;

enum { ORC_PROBE_M = 0, ORC_PROBE_H = 1, ORC_PROBE_N = 2, ORC_PROBE_SYN_G = 3, ORC_PROBE_TIME = 4,
       ORC_PROBE_NSTEPS = 5 };

/* ---- building blocks, exported so the tests can pin each one separately ---- */
double orc_exprelr(double x);                       /* x/expm1(x), 1 at x == 0            */
void orc_hh_rates(double v, double out[6]);         /* am, bm, ah, bh, an, bn  [1/ms]     */
/* d_i = C_i/dt + sum_j sigma_ij, u_i = -sigma_{i,parent}, rhs_i = C_i/dt V_i - I_i */
void orc_assemble(int64_t n, const int32_t* parent, const double* area, const double* cm,
                  const double* raxial, const double* v, const double* i_memb, double delta,
                  double* d, double* u, double* rhs);
/* Hines / extended Thomas solve; d and rhs are overwritten, x receives V' */
void orc_hines_solve(int64_t n, const int32_t* parent, double* d, const double* u, double* rhs,
                     double* x);

/* ---- the model ---- */
int orc_create(const orc_desc* desc, orc_model** out);       /* 0 or negative error code      */
int orc_advance(orc_model* m, double t_end, double dt);
int64_t orc_spikes(orc_model* m, int64_t* cell, double* time, int64_t cap); /* sorted (time,cell) */
int orc_voltage(orc_model* m, double* out, int64_t n_cv);
int orc_probe(orc_model* m, int what, double* out, int64_t n);
/* membrane current I_i [nA] of every CV of one cell at the model's current state and time */
int orc_cell_currents(orc_model* m, int64_t cell, double* i_out);
/* overwrite the state (any pointer may be NULL) and reset the detector history (armed, v_prev):
 * used by the parity tests to start both implementations from one state */
int orc_set_state(orc_model* m, const double* v, const double* hm, const double* hh,
                  const double* hn, const double* syn_g);
/* 0 (default): explicit membrane currents, the equation at PAPER.md:154 (reading R1).  1: the conductance-
 * linearised variant: membrane conductances on the diagonal, matrix assembled and
 * eliminated every step. */
int orc_set_linearised(orc_model* m, int on);
void orc_set_threads(int n);                                  /* OpenMP threads (timing only)  */
int orc_get_threads(void);
void orc_destroy(orc_model* m);
const char* orc_last_error(void);

#ifdef __cplusplus
}
#endif
#endif
