/* Tier W of the CPU oracle: brute-force Wick contraction of the interpolating operators.
 *
 * TEST INFRASTRUCTURE ONLY (see oracle/nbs_oracle.py header).  Shares no code with the CUDA path.
 *
 * What it computes (eq. 2.1 with the operators of PAPER.md:33-41 eqs. 2.2-2.3 and the
 * source weights of PAPER.md:45 eq. 2.4), with no baryon blocks and no permutation bookkeeping:
 *
 *   F_{a1 a2 a3 a4}(r) = sum_X sum_{terms} k1 k2 k3 k4
 *        sum_{eta1..eta6, xi'1..xi'6} W[eta1 eta2 eta3; a1] W[eta4 eta5 eta6; a2]
 *                                    W[xi'1 xi'2 xi'3; a3] W[xi'4 xi'5 xi'6; a4]
 *        < q_f1(X+r,eta1) q_f2(X+r,eta2) q_f3(X+r,eta3) q_f4(X,eta4) q_f5(X,eta5) q_f6(X,eta6)
 *          qbar_h6(xi'6) ... qbar_h1(xi'1) >
 *
 * and the fermion expectation value is the determinant of the 6x6 matrix
 *   M[j][k] = delta(f_j, h_k) S_{f_j}(x_j)[eta_j][xi'_k]          (Wick's theorem; the nested
 * ordering q_1..q_6 qbar_6..qbar_1 gives the identity pairing sign +1).
 * W[xi1 xi2 xi3; a] = eps_{c1c2c3} (C g5)_{a1 a2} delta_{a3 a}, xi = colour + 3 spin.
 * Only the 24 non-zero entries of each W are visited: 24^4 determinants per site pair, spin
 * combination and term combination.
 */
#include <complex.h>
#include <math.h>
#include <stdlib.h>
#include <string.h>

typedef double complex cplx;

static const double CG5[4][4] = {{0, 1, 0, 0}, {-1, 0, 0, 0}, {0, 0, 0, 1}, {0, 0, -1, 0}};

static double eps3(int a, int b, int c) {
    if (a == b || b == c || a == c) return 0.0;
    return ((b - a) * (c - a) * (c - b) > 0) ? 1.0 : -1.0;
}

/* non-zeros of W[.;a]: 24 of them */
static int w_nonzeros(int a, int idx[24][3], double val[24]) {
    int n = 0;
    for (int c1 = 0; c1 < 3; c1++)
        for (int c2 = 0; c2 < 3; c2++)
            for (int c3 = 0; c3 < 3; c3++)
                for (int a1 = 0; a1 < 4; a1++)
                    for (int a2 = 0; a2 < 4; a2++) {
                        double w = eps3(c1, c2, c3) * CG5[a1][a2];
                        if (w == 0.0) continue;
                        idx[n][0] = c1 + 3 * a1;
                        idx[n][1] = c2 + 3 * a2;
                        idx[n][2] = c3 + 3 * a;
                        val[n] = w;
                        n++;
                    }
    return n;
}

/* determinant by Gaussian elimination with partial pivoting */
static cplx det6(cplx M[6][6]) {
    cplx det = 1.0;
    for (int c = 0; c < 6; c++) {
        int piv = c;
        double best = cabs(M[c][c]);
        for (int r = c + 1; r < 6; r++) {
            double v = cabs(M[r][c]);
            if (v > best) { best = v; piv = r; }
        }
        if (best == 0.0) return 0.0;
        if (piv != c) {
            for (int k = 0; k < 6; k++) { cplx t = M[c][k]; M[c][k] = M[piv][k]; M[piv][k] = t; }
            det = -det;
        }
        det *= M[c][c];
        cplx inv = 1.0 / M[c][c];
        for (int r = c + 1; r < 6; r++) {
            cplx f = M[r][c] * inv;
            if (f == 0.0) continue;
            for (int k = c + 1; k < 6; k++) M[r][k] -= f * M[c][k];
        }
    }
    return det;
}

/* One site pair.  S[f] -> [12][12] matrices at x (rows 0-2) and y (rows 3-5).
 * f[6]: flavours (0,1,2 = u,d,s) of the six sink quark fields; h[6]: of the six source quarks. */
static cplx pair_term(const cplx* Sx[3], const cplx* Sy[3], const int f[6], const int h[6],
                      int a1, int a2, int a3, int a4) {
    int i1[24][3], i2[24][3], i3[24][3], i4[24][3];
    double v1[24], v2[24], v3[24], v4[24];
    w_nonzeros(a1, i1, v1);
    w_nonzeros(a2, i2, v2);
    w_nonzeros(a3, i3, v3);
    w_nonzeros(a4, i4, v4);
    cplx acc = 0.0;
    for (int n3 = 0; n3 < 24; n3++)
        for (int n4 = 0; n4 < 24; n4++) {
            int xs[6] = {i3[n3][0], i3[n3][1], i3[n3][2], i4[n4][0], i4[n4][1], i4[n4][2]};
            for (int n1 = 0; n1 < 24; n1++)
                for (int n2 = 0; n2 < 24; n2++) {
                    int et[6] = {i1[n1][0], i1[n1][1], i1[n1][2], i2[n2][0], i2[n2][1], i2[n2][2]};
                    cplx M[6][6];
                    for (int j = 0; j < 6; j++) {
                        const cplx* S = (j < 3) ? Sx[f[j]] : Sy[f[j]];
                        for (int k = 0; k < 6; k++)
                            M[j][k] = (f[j] == h[k]) ? S[et[j] * 12 + xs[k]] : 0.0;
                    }
                    acc += v1[n1] * v2[n2] * v3[n3] * v4[n4] * det6(M);
                }
        }
    return acc;
}

/* F[r][ispin] for the listed spin combinations.
 * S_u, S_d, S_s: [V][12][12] complex128 (interleaved), site = x + L (y + L z).
 * Baryon i (i=0..3 for B1..B4) is sum_t coef[i][t] * E[flav[i][t][0..2]], nterm[i] terms (<= 3).
 * spins: [nspin][4] = (a1,a2,a3,a4).  rlist: r values to evaluate (nr of them); F: [nr][nspin]. */
int wick_fourpt(int L, const double* S_u, const double* S_d, const double* S_s,
                const int* nterm, const double* coef, const int* flav,
                int nspin, const int* spins, int nr, const int* rlist, double* F_out) {
    const int V = L * L * L;
    const cplx* S[3] = {(const cplx*)S_u, (const cplx*)S_d, (const cplx*)S_s};
    cplx* F = (cplx*)F_out;
    memset(F, 0, sizeof(cplx) * (size_t)nr * nspin);
    /* one work item per (r, spin combination, X): a flat loop so that a single (r, spin) request
     * still uses every core */
    const long nitem = (long)nr * nspin * V;
#pragma omp parallel for schedule(dynamic)
    for (long item = 0; item < nitem; item++) {
        int X = (int)(item % V);
        int is = (int)((item / V) % nspin);
        int ir = (int)(item / ((long)V * nspin));
        int r = rlist[ir];
        int rx = r % L, ry = (r / L) % L, rz = r / (L * L);
        int x0 = X % L, y0 = (X / L) % L, z0 = X / (L * L);
        int xs = ((x0 + rx) % L) + L * (((y0 + ry) % L) + L * ((z0 + rz) % L));
        const cplx* Sx[3] = {S[0] + (size_t)xs * 144, S[1] + (size_t)xs * 144, S[2] + (size_t)xs * 144};
        const cplx* Sy[3] = {S[0] + (size_t)X * 144, S[1] + (size_t)X * 144, S[2] + (size_t)X * 144};
        cplx acc = 0.0;
        for (int t1 = 0; t1 < nterm[0]; t1++)
            for (int t2 = 0; t2 < nterm[1]; t2++)
                for (int t3 = 0; t3 < nterm[2]; t3++)
                    for (int t4 = 0; t4 < nterm[3]; t4++) {
                        int f[6], h[6];
                        for (int m = 0; m < 3; m++) {
                            f[m] = flav[(0 * 3 + t1) * 3 + m];
                            f[3 + m] = flav[(1 * 3 + t2) * 3 + m];
                            h[m] = flav[(2 * 3 + t3) * 3 + m];
                            h[3 + m] = flav[(3 * 3 + t4) * 3 + m];
                        }
                        double k = coef[0 * 3 + t1] * coef[1 * 3 + t2] * coef[2 * 3 + t3] * coef[3 * 3 + t4];
                        acc += k * pair_term(Sx, Sy, f, h, spins[is * 4 + 0], spins[is * 4 + 1],
                                             spins[is * 4 + 2], spins[is * 4 + 3]);
                    }
        double* dst = (double*)&F[(size_t)ir * nspin + is];
#pragma omp atomic
        dst[0] += creal(acc);
#pragma omp atomic
        dst[1] += cimag(acc);
    }
    return 0;
}
