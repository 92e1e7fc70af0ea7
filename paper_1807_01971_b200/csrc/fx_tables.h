// fx_tables.h -- fp64 reference-element tables shared by fx_tables.cpp (host, g++) and fx.cu (nvcc).
#ifndef FX_TABLES_H
#define FX_TABLES_H

#define FX_PMAX 5

typedef struct {
    int P;
    double xi[FX_PMAX], w[FX_PMAX];          // Gauss-Legendre nodes (ascending) and weights on [-1,1]
    double L[FX_PMAX], R[FX_PMAX];           // l_m(-1), l_m(+1)
    double B[FX_PMAX];                       // R[k]/w[k]
    double T0[FX_PMAX][FX_PMAX];             // D[k][m] - R[k]R[m]/w[k]
    double T0L[FX_PMAX][FX_PMAX];            // T0 + L[k]L[m]/w[k]     (first cell of a Dirichlet direction)
    double WW[FX_PMAX][FX_PMAX];             // w[l]*w[k]
    double D[FX_PMAX][FX_PMAX];              // l_m'(xi_k)
} fx_tables;

#ifdef __cplusplus
extern "C"
#endif
int fx_make_tables(int P, fx_tables* t);

#endif
