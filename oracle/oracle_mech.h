/* oracle/oracle_mech.h -- the CPU oracle's own description of a kinetic model.
 *
 * TEST INFRASTRUCTURE ONLY.  Nothing under oracle/ is part of the product path: only
 * tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may load it.  It shares no code, header, table or helper with the CUDA library.
 *
 * All pointers are HOST pointers owned by the caller and only read during a call.
 * Field meaning follows PAPER.md Sections 2.2-2.3 (see each function in oracle.c for
 * the equation it implements).  Units: SI with kmol.
 */
#ifndef ORACLE_MECH_H
#define ORACLE_MECH_H

typedef struct {
    int ns;                    /* N_sp  */
    int nr;                    /* N_reac */
    const double *mw;          /* [ns]      W_k, kg/kmol (Eq. 4) */
    const double *nasa_lo;     /* [ns][7]   a_0..a_6 for T <= t_mid (Eqs. 9-11) */
    const double *nasa_hi;     /* [ns][7]   a_0..a_6 for T >  t_mid */
    const double *t_mid;       /* [ns] */
    const int *reac_ptr, *reac_spec, *reac_nu;   /* CSR: nu'_ki  (Eq. 15) */
    const int *prod_ptr, *prod_spec, *prod_nu;   /* CSR: nu''_ki */
    const int *rxn_type;       /* [nr] 0 elementary, 1 third-body, 2 falloff, 3 chem.-activated,
                                       4 PLOG, 5 Chebyshev  (Eq. 20, Eqs. 37-43) */
    const int *rev_type;       /* [nr] 0 irreversible, 1 k_r = k_f/K_c (Eq. 23), 2 explicit */
    const double *arr_hi;      /* [nr][3] A, beta, Ta (Eq. 21); k_inf for types 2, 3 */
    const double *arr_lo;      /* [nr][3] k_0 for types 2, 3 */
    const double *arr_rev;     /* [nr][3] explicit reverse parameters */
    const int *falloff_form;   /* [nr] 0 Lindemann, 1 Troe, 2 SRI (Eq. 32) */
    const double *falloff_par; /* [nr][5] Troe: a, T***, T*, T**, has_T**;  SRI: a, b, c, d, e */
    const int *tb_species;     /* [nr] m >= 0: [X]_i = [X_m] (Eq. 30); -1: mixture (Eq. 28) */
    const int *eff_ptr, *eff_spec;               /* CSR: alpha_ij where != 1 */
    const double *eff_val;
    const int *plog_ptr;       /* [nr+1] */
    const double *plog_p;      /* Pa, ascending within a reaction */
    const double *plog_arr;    /* [][3] A, beta, Ta at each pressure (Eqs. 37-38) */
    const int *cheb_ptr;       /* [nr+1] offsets into cheb_eta */
    const int *cheb_nT, *cheb_nP;
    const double *cheb_lim;    /* [nr][4] Tmin, Tmax, pmin, pmax (Eqs. 42-43) */
    const double *cheb_eta;    /* eta_ij, row-major in (i, j) (Eq. 40) */
} orc_mech;

#endif
