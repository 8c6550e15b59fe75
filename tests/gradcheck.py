"""The gradient parity check shared by tests/test_gpu_raster.py and __graft_entry__.smoke() (reading G-4).

BASELINE.json north_star: "Gradients must agree within 1e-3 relative (1e-5 abs floor)". Every gradient element is a sum
of thousands of signed per-pixel products accumulated in fp32 in an order the atomics choose; no fp32 summation (in any
order) can be held to less than a small multiple of 2^-24 * sum|product|. So the bound asserted for 100 % of the
elements of every gradient array is

    |gpu - oracle| <= max(1e-3 |oracle|, 1e-5, C_COND * 2^-24 * abs_sum)

where abs_sum is the oracle's sum of the absolute values of the products behind that element (its conditioning, pushed
through |J| of the projection backward for the 3D parameters; oracle/legs_oracle.py::render_backward(with_abs=True)).
C_COND is ONE constant for every array, scene and size. Elements that need the third term are counted and the worst
ones are listed with their condition number abs_sum / |oracle| ("listed separately with their
condition number rather than silently dropped").

Derivation of C_COND (G-4): a product is evaluated in fp32 through ~12 roundings (pixel offset, the two
whitened coordinates, the exponent, ex2.approx at 2 ulp, alpha, the weight alpha*T, the upstream factor, the geometry
factor) plus one rounding per blended Gaussian behind it for the transmittance chain T_k = T_final / prod (1 - alpha_j)
(tens of factors at the pixel counts of the configs); signed roundings add like a random walk, so a product is good to
a few 2^-24 and the fp32 accumulation (32-lane butterfly, then one atomic per warp) adds log2(32) more: a budget of ~8.
Measured (round 2, every scene family and full size): need_c <= 0.7, on at most 12 elements per array, all with condition
numbers above 4e4. Round 3 asserts that instead of printing it: C_COND = 4, and per array at most
MAX_CONDITIONED = 32 elements may need the third term at all, none of them more than MAX_NEED_C = 3 (measured in round 3
over the 33 gradient tests: at most 6 elements per array, need_c <= 1.31, condition numbers 1.9e4 .. 1.5e7; the atomics'
order varies from run to run, hence the slack), so the relaxation of north_star's bound is itself bounded by the test. abs_sum is pinned independently of the
gradients in tests/test_oracle_conditioning.py (triangle inequality, one-signed sums, explicit numpy expansion, |J| by central
differences).
"""
import numpy as np

GRAD_KEYS = ("dmeans", "dscales", "dquats", "dopacities", "dsh", "dsem", "dunc", "dmean2d")
REL, FLOOR = 1e-3, 1e-5          # north_star
C_COND = 4.0
MAX_CONDITIONED = 32      # elements per array that may need the conditioning term at all
MAX_NEED_C = 3.0          # and the largest multiple of 2^-24 abs_sum any of them may need
EPS = 2.0 ** -24


def check_grads(gpu: dict, ref: dict, verbose: bool = True) -> dict:
    """gpu[k]: arrays from the CUDA path; ref[k]: oracle gradients, ref["abs"][k]: their absolute sums.
    Asserts the bound above for every element. Returns per array: (elements needing the conditioning term, the c that
    would have been needed, worst condition number among them)."""
    report = {}
    for k in GRAD_KEYS:
        a = np.asarray(gpu[k], dtype=np.float64).reshape(-1)
        b = np.asarray(ref[k], dtype=np.float64).reshape(-1)
        s = np.asarray(ref["abs"][k], dtype=np.float64).reshape(-1)
        err = np.abs(a - b)
        strict = np.maximum(REL * np.abs(b), FLOOR)
        bound = np.maximum(strict, C_COND * EPS * s)
        beyond = err > strict
        need_c = float((err[beyond] / (EPS * np.maximum(s[beyond], 1e-300))).max()) if beyond.any() else 0.0
        worst_cond = float((s[beyond] / np.maximum(np.abs(b[beyond]), 1e-300)).max()) if beyond.any() else 0.0
        report[k] = dict(n=int(a.size), conditioned=int(beyond.sum()), need_c=round(need_c, 2), worst_cond=worst_cond)
        bad = err > bound
        if verbose and beyond.any():
            idx = np.flatnonzero(beyond)
            idx = idx[np.argsort(-(err[idx] / strict[idx]))[:3]]
            for i in idx:
                print(f"  G-4 {k}[{i}]: ref {b[i]:+.3e} gpu {a[i]:+.3e} err {err[i]:.2e} cond {s[i] / max(abs(b[i]), 1e-300):.1e} "
                      f"needs c = {err[i] / (EPS * max(s[i], 1e-300)):.1f}")
        assert not bad.any(), (f"{k}: {int(bad.sum())} of {a.size} elements beyond max(1e-3|ref|, 1e-5, {C_COND:g} 2^-24 sum|term|); "
                               f"worst needs c = {need_c:.1f}")
        assert int(beyond.sum()) <= MAX_CONDITIONED, (f"{k}: {int(beyond.sum())} of {a.size} elements need the conditioning term "
                                                      f"(more than {MAX_CONDITIONED}: the strict 1e-3 / 1e-5 bound must hold nearly everywhere)")
        assert need_c <= MAX_NEED_C, f"{k}: an element needs c = {need_c:.2f} > {MAX_NEED_C:g}"
    return report
