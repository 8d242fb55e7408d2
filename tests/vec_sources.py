"""User integrands for the vector-valued tests (R15): plain C++ text that is valid CUDA device code AND valid
host C++ (with `__device__` defined away), so that NVRTC and g++ compile the very same text. They are INPUTS of the
method, like integrand parameters. Only + - * (and fmaf where a built-in is restated) are used where bit-exact
agreement between the two sides is asserted: with --fmad=false / -ffp-contract=off both sides round identically."""

_PAIR = """
__device__ void %(name)s(const float* x, int dim, const float* p, int np, float* out, int n_out) { %(name)s_t<float>(x, dim, p, np, out, n_out); }
__device__ void %(name)s(const double* x, int dim, const double* p, int np, double* out, int n_out) { %(name)s_t<double>(x, dim, p, np, out, n_out); }
"""


def _templated(name, body):
    return ("template <class R> __device__ inline void %s_t(const R* x, int dim, const R* p, int np, R* out, int n_out) {\n%s\n}\n"
            % (name, body)) + _PAIR % {"name": name}


# LINEAR restated operation by operation (R8): FP64 p0 + sum (p_d * x_d) with separate roundings; FP32 fmaf chain
LINEAR1 = """
__device__ void lin1(const double* x, int dim, const double* p, int np, double* out, int n_out) {
    double f = p[0];
    for (int d = 0; d < dim; ++d) { double t = p[1 + d] * x[d]; f = f + t; }
    out[0] = f;
}
__device__ void lin1(const float* x, int dim, const float* p, int np, float* out, int n_out) {
    float f = p[0];
    for (int d = 0; d < dim; ++d) f = fmaf(p[1 + d], x[d], f);
    out[0] = f;
}
"""

# SIN_SUM in FP64 through the platform's sin (oracle-side pin only: libm there, libdevice on the GPU)
SIN1 = """
__device__ void sin1(const double* x, int dim, const double* p, int np, double* out, int n_out) {
    double a = x[0];
    for (int d = 1; d < dim; ++d) a = a + x[d];
    out[0] = sin(a);
}
"""

# four polynomial components over a 3-D box: closed forms 2, 4/3, 12, 2 over [0,1]x[0,2]x[-1,1]
POLY4 = _templated("poly4", """
    out[0] = x[0] * x[1];
    out[1] = x[2] * x[2];
    out[2] = R(3);
    R t = x[1] * x[2];
    out[3] = x[0] + t;""")

# two components that vary along different axes, and each of them alone
TWO_AXES = _templated("two_axes", """
    out[0] = x[0] * x[0];
    R t = x[1] * x[1];
    out[1] = t * x[1];""")
AXIS0 = _templated("axis0", "    out[0] = x[0] * x[0];")
AXIS1 = _templated("axis1", """
    R t = x[1] * x[1];
    out[0] = t * x[1];""")
AXIS0_TWICE = _templated("axis0_twice", """
    out[0] = x[0] * x[0];
    out[1] = x[0] * x[0];""")

# per-instance parameter p[0] scales both components (a parameter sweep over a vector-valued function)
SCALED_AXES = _templated("scaled_axes", """
    R a = x[0] * x[0];
    out[0] = p[0] * a;
    R t = x[1] * x[1];
    R b = t * x[1];
    out[1] = p[0] * b;""")

# eight polynomial moments of s = p0 * sum_d x_d sharing one sample stream: the bench's vector-valued workload (an input recipe,
# kept with the other workloads)
from paper_1902_07916_b200.workloads import VEC_MOMENTS_SRC as MOMENTS8  # noqa: E402
