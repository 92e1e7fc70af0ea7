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

// stand-alone derivative y <- alpha M x + beta y: per flux (0 forward, 1 backward, 2 centred)
typedef struct {
    double TT[2][FX_PMAX][FX_PMAX];          // [0] interior cell, [1] first cell of a Dirichlet line
    double cN[FX_PMAX], cP[FX_PMAX];         // coefficients of the next cell's left trace / previous cell's right trace
} fx_dtables;

#ifdef __cplusplus
extern "C" {
#endif
int fx_make_tables(int P, fx_tables* t);
int fx_make_dtables(int P, int flux, fx_dtables* d);
#ifdef __cplusplus
}
#endif

#endif
