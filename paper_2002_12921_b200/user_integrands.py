"""CUDA sources of user-supplied integrands for vegas_set_user_integrand (include/vegas.h): the streaming form
`struct vegas_user_integrand { begin(dim, p); dim(j, x, p); finish(p); }` the fused kernel is compiled around.

These are examples that ship with the library and the inputs of the user-integrand parity tests; each states the
formula it implements.  Parameters are the same host arrays the built-in integrands take (the top-level `workloads` module).
"""

# PAPER.md:69 Eq.(2) as printed, N = 1: f = 0 if any x_j <= a_j, else exp(sum_j c_j x_j); p = { c[0..d-1], a[0..d-1] }
GENZ_DISCONTINUOUS = r"""
struct vegas_user_integrand {
    double s;
    int d;
    bool zero;
    __device__ void begin(int dim, const double* p) { s = 0.0; d = dim; zero = false; }
    __device__ void dim(int j, double x, const double* p) {
        zero = zero || (x <= p[d + j]);
        s = fma(p[j], x, s);
    }
    __device__ double finish(const double* p) { return zero ? 0.0 : exp(s); }
};
"""

# PAPER.md:65 Eq.(1): (a sqrt(pi))^-d exp(-sum_j (x_j - 1/2)^2 / a^2); p = { a }
GAUSS = r"""
struct vegas_user_integrand {
    double s;
    int d;
    __device__ void begin(int dim, const double* p) { s = 0.0; d = dim; }
    __device__ void dim(int j, double x, const double* p) { const double t = x - 0.5; s = fma(t, t, s); }
    __device__ double finish(const double* p) {
        const double a = p[0];
        return pow(a * sqrt(3.14159265358979323846), -(double)d) * exp(-s / (a * a));
    }
};
"""

# PAPER.md:74 Eq.(3), N = 1: prod_j 1/(c_j^-2 + (x_j - w_j)^2); p = { c[0..d-1], w[0..d-1] }
GENZ_PRODUCT_PEAK = r"""
struct vegas_user_integrand {
    double prod;
    int d;
    __device__ void begin(int dim, const double* p) { prod = 1.0; d = dim; }
    __device__ void dim(int j, double x, const double* p) {
        const double t = x - p[d + j];
        prod *= 1.0 / (p[j] * p[j]) + t * t;
    }
    __device__ double finish(const double* p) { return 1.0 / prod; }
};
"""

# does not compile: the error path of vegas_set_user_integrand (tests)
BROKEN = r"""
struct vegas_user_integrand {
    __device__ void begin(int dim, const double* p) { undeclared_symbol = 1; }
    __device__ void dim(int j, double x, const double* p) {}
    __device__ double finish(const double* p) { return 1.0; }
};
"""

# Eq.(3) again, with an observable: the coordinate x_{d-1}, histogrammed with weight f*J during the
# integration (vegas_set_observable / vegas_get_observable_hist)
GENZ_PRODUCT_PEAK_WITH_OBSERVABLE = r"""
struct vegas_user_integrand {
    double prod, xlast;
    int d;
    __device__ void begin(int dim, const double* p) { prod = 1.0; d = dim; xlast = 0.0; }
    __device__ void dim(int j, double x, const double* p) {
        const double t = x - p[d + j];
        prod *= 1.0 / (p[j] * p[j]) + t * t;
        if (j == d - 1) xlast = x;
    }
    __device__ double finish(const double* p) { return 1.0 / prod; }
    __device__ double observable(const double* p) { return xlast; }
};
"""
