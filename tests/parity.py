"""Error measures and tolerances of the GPU-vs-oracle parity tests (test helper, not product).

BASELINE.json north_star fixes the bar; SURVEY.md 8(c) reading 12 fixes the measure:
  acc   per particle |a_gpu - a_ref|_2 / |a_ref|_2   <= 1e-4 at the 99th percentile, <= 1e-2 max
  jerk  per particle |j_gpu - j_ref|_2 / |j_ref|_2   <= 1e-3 at the 99th percentile
  pot   per particle |p_gpu - p_ref| / |p_ref|       <= 1e-5 (max)
"""
import numpy as np

ACC_P99, ACC_MAX, JERK_P99, POT_MAX = 1e-4, 1e-2, 1e-3, 1e-5


def vec_rel_err(got, ref):
    got = np.asarray(got, dtype=np.float64)
    ref = np.asarray(ref, dtype=np.float64)
    num = np.sqrt(np.sum((got - ref) ** 2, axis=1))
    den = np.sqrt(np.sum(ref ** 2, axis=1))
    return num / np.where(den > 0.0, den, 1.0)


def scalar_rel_err(got, ref):
    got = np.asarray(got, dtype=np.float64)
    ref = np.asarray(ref, dtype=np.float64)
    return np.abs(got - ref) / np.where(ref != 0.0, np.abs(ref), 1.0)


def errors(got, ref, jerk=True):
    acc, jrk, pot = got
    racc, rjrk, rpot = ref
    ea = vec_rel_err(acc, racc)
    out = dict(acc_p99=float(np.percentile(ea, 99)) if ea.size else 0.0,
               acc_max=float(ea.max()) if ea.size else 0.0)
    ep = scalar_rel_err(pot, rpot)
    out["pot_max"] = float(ep.max()) if ep.size else 0.0
    if jerk:
        ej = vec_rel_err(jrk, rjrk)
        out["jerk_p99"] = float(np.percentile(ej, 99)) if ej.size else 0.0
        out["jerk_max"] = float(ej.max()) if ej.size else 0.0
    return out


def assert_parity(got, ref, jerk=True, what=""):
    e = errors(got, ref, jerk)
    assert np.all(np.isfinite(got[0])) and np.all(np.isfinite(got[2])), f"{what}: non-finite result"
    assert e["acc_p99"] <= ACC_P99, f"{what}: acc p99 {e['acc_p99']:.3e} > {ACC_P99}"
    assert e["acc_max"] <= ACC_MAX, f"{what}: acc max {e['acc_max']:.3e} > {ACC_MAX}"
    assert e["pot_max"] <= POT_MAX, f"{what}: pot max {e['pot_max']:.3e} > {POT_MAX}"
    if jerk:
        assert np.all(np.isfinite(got[1])), f"{what}: non-finite jerk"
        assert e["jerk_p99"] <= JERK_P99, f"{what}: jerk p99 {e['jerk_p99']:.3e} > {JERK_P99}"
    return e
