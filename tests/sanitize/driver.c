/* Driver for the sanitizer build of the oracles (tests/test_oracle_sanitizers.py): calls every exported entry point on
 * small seeded inputs, all four boundary mixes, so that AddressSanitizer / UBSan see every loop of oracle/*.c. */
#include <stdio.h>
#include <stdlib.h>
#include <math.h>

int oracle_pressure_projection(int, int, int, double, double, const double*, int, int, double*, double*, double*, double*, double*, double, double);
int oracle_laplacian(int, int, int, double, double, const double*, int, int, const double*, double*);
int oracle_dft(int, int, const double*, const double*, double*, double*);
int oracle_dct(int, int, const double*, double*);
int oracle_gauge_column(int, const double*, const double*, double*);
int oracle_viscous_step(int, int, int, double, double, const double*, int, int, double*, double*, double*, const double*, const double*, const double*, double);
int oracle_cyclic_thomas(int, const double*, const double*, const double*, const double*, double*);
int oracle_explicit_terms(int, int, int, double, double, const double*, int, int, const double*, const double*, const double*, const double*,
                          const double*, const double*, const double*, double*, double*, double*, double*, double*, double*, double, double, double, double);
int oracle_mls_interpolate(int, int, int, double, double, const double*, int, int, long, const double*, const double*, const double*,
                           const double*, const double*, const double*, double*, double*, double*);
int oracle_ibm_forcing(int, int, int, double, double, const double*, int, int, long, const double*, const double*, const double*, const double*,
                       const double*, const double*, const double*, const double*, const double*, const double*, double,
                       double*, double*, double*, double*, double*, double*);

static unsigned long long st = 88172645463325252ULL;
static double rnd(void) { st ^= st << 13; st ^= st >> 7; st ^= st << 17; return (double)(st >> 11) / 9007199254740992.0 - 0.5; }
static double* field(size_t n) { double* p = malloc(sizeof(double) * n); for (size_t i = 0; i < n; i++) p[i] = rnd(); return p; }

int main(void)
{
    const int shapes[3][3] = {{8, 6, 7}, {12, 4, 5}, {6, 6, 9}};
    int bad = 0;
    for (int sh = 0; sh < 3; sh++)
        for (int bc = 0; bc < 4; bc++) {
            const int nx = shapes[sh][0], ny = shapes[sh][1], nz = shapes[sh][2], bx = bc & 1, by = bc >> 1;
            const size_t N = (size_t)nx * ny * nz;
            double* zc = malloc(sizeof(double) * (nz + 1));
            for (int k = 0; k <= nz; k++) zc[k] = 0.5 * (1.0 + tanh(2.0 * (2.0 * k / nz - 1.0)) / tanh(2.0));
            double *u = field(N), *v = field(N), *w = field(N), *p = field(N), *phi = field(N);
            double *hu = field(N), *hv = field(N), *hw = field(N), *ru = field(N), *rv = field(N), *rw = field(N);
            for (int j = 0; j < ny; j++) for (int i = 0; i < nx; i++) w[(size_t)j * nx + i] = 0.0;
            bad |= oracle_explicit_terms(nx, ny, nz, 1.0, 1.5, zc, bx, by, u, v, w, p, hu, hv, hw, hu, hv, hw, ru, rv, rw, 1.5e-3, -0.5e-3, 1e-3, 1e-4);
            bad |= oracle_viscous_step(nx, ny, nz, 1.0, 1.5, zc, bx, by, u, v, w, ru, rv, rw, 0.3);
            bad |= oracle_pressure_projection(nx, ny, nz, 1.0, 1.5, zc, bx, by, u, v, w, p, phi, 1e-3, 1e-4);
            bad |= oracle_laplacian(nx, ny, nz, 1.0, 1.5, zc, bx, by, phi, ru);
            const long nm = 40;
            double *xm = field(nm), *ym = field(nm), *zm = field(nm), *ar = field(nm), *F0 = field(nm), *F1 = field(nm), *F2 = field(nm);
            for (long l = 0; l < nm; l++) { xm[l] += 0.5; ym[l] = 1.5 * (ym[l] + 0.5); zm[l] += 0.5; }
            if (nx >= 3 && ny >= 3) {
                bad |= oracle_mls_interpolate(nx, ny, nz, 1.0, 1.5, zc, bx, by, nm, xm, ym, zm, u, v, w, F0, F1, F2);
                bad |= oracle_ibm_forcing(nx, ny, nz, 1.0, 1.5, zc, bx, by, nm, xm, ym, zm, ar, F0, F1, F2, u, v, w, 100.0, F0, F1, F2, hu, hv, hw);
            }
            bad |= oracle_gauge_column(nz, zc, u, v);
            free(zc); free(u); free(v); free(w); free(p); free(phi); free(hu); free(hv); free(hw); free(ru); free(rv); free(rw);
            free(xm); free(ym); free(zm); free(ar); free(F0); free(F1); free(F2);
        }
    for (int n = 1; n <= 30; n++) {
        double *a = field(n), *b = field(n), *c = field(n), *d = field(n), *x = field(n), *y = field(n);
        for (int i = 0; i < n; i++) b[i] = 3.0 + fabs(a[i]) + fabs(c[i]);
        bad |= oracle_cyclic_thomas(n, a, b, c, d, x);
        bad |= oracle_dft(n, -1, a, c, x, y);
        bad |= oracle_dct(n, n & 1, a, x);
        free(a); free(b); free(c); free(d); free(x); free(y);
    }
    printf("sanitizer driver done, status %d\n", bad);
    return bad ? 1 : 0;
}
