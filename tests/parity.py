"""The three-class parity rule of DESIGN.md §4, used by every GPU-vs-oracle test.

north_star's tolerance, verbatim: |gpu - oracle| <= max(1e-4 * |oracle|, 1e-6). It applies unchanged
to STRICT individuals (those whose certified fp32 error bound E_p is far below it). CONDITIONED
individuals (ill-conditioned programs: E_p comparable to or above the tolerance) get the tolerance
plus 2*E_p. UNSTABLE / CLASS_UNSTABLE individuals (an intermediate straddles a protected-operator
threshold or the fp32 overflow edge) are exempt from value and class parity and only counted.
Class parity (finite / +inf / NaN) is exact for every other individual; malformed individuals must
be the canonical quiet NaN bit pattern.
"""
import numpy as np

RTOL = 1e-4   # north_star
ATOL = 1e-6   # north_star

FLAG_MALFORMED, FLAG_UNSTABLE, FLAG_CLASS_UNSTABLE = 1, 2, 4


def klass(f):
    """0 finite, 1 +inf, 2 -inf, 3 NaN."""
    f = np.asarray(f, np.float32)
    return np.where(np.isnan(f), 3, np.where(np.isposinf(f), 1, np.where(np.isneginf(f), 2, 0)))


def compare(gpu, orc):
    """gpu: float32[P]; orc: dict from oracle.binding.evaluate. Returns a report dict; report['bad']
    lists the indices that violate the rule."""
    gpu = np.asarray(gpu, np.float32)
    fo = orc["fitness"].astype(np.float32)
    E = orc["bound"].astype(np.float64)
    flags = orc["flags"]
    P = gpu.shape[0]
    malformed = (flags & FLAG_MALFORMED) != 0
    exempt = ((flags & (FLAG_UNSTABLE | FLAG_CLASS_UNSTABLE)) != 0) & ~malformed
    checked = ~malformed & ~exempt

    bad = np.zeros(P, bool)
    # malformed: canonical quiet NaN, bit exact
    bad |= malformed & (gpu.view(np.uint32) != np.uint32(0x7FC00000))
    # class parity, exact
    kg, ko = klass(gpu), klass(fo)
    class_bad = checked & (kg != ko)
    bad |= class_bad
    # value parity on finite individuals
    fin = checked & (ko == 0) & (kg == 0)
    with np.errstate(all="ignore"):
        diff = np.abs(gpu.astype(np.float64) - fo.astype(np.float64))
        tol = np.maximum(RTOL * np.abs(fo.astype(np.float64)), ATOL)
    strict = fin & (2.0 * E <= 0.5 * tol)
    cond = fin & ~strict
    strict_bad = strict & ~(diff <= tol)
    cond_bad = cond & ~(diff <= tol + 2.0 * E)
    bad |= strict_bad | cond_bad
    with np.errstate(all="ignore"):
        rel = np.where(fin, diff / np.maximum(np.abs(fo.astype(np.float64)), 1e-30), 0.0)
    return dict(P=P, strict=int(strict.sum()), conditioned=int(cond.sum()), exempt=int(exempt.sum()),
                malformed=int(malformed.sum()), invalid=int((checked & (ko != 0)).sum()),
                class_bad=int(class_bad.sum()), strict_bad=int(strict_bad.sum()),
                cond_bad=int(cond_bad.sum()), bad=np.nonzero(bad)[0],
                max_rel_strict=float(rel[strict].max()) if strict.any() else 0.0)


def describe(rep, gpu, orc, limit=8):
    lines = [f"P={rep['P']} strict={rep['strict']} conditioned={rep['conditioned']} "
             f"exempt={rep['exempt']} malformed={rep['malformed']} invalid={rep['invalid']} "
             f"class_bad={rep['class_bad']} strict_bad={rep['strict_bad']} cond_bad={rep['cond_bad']} "
             f"max_rel_strict={rep['max_rel_strict']:.3g}"]
    for i in rep["bad"][:limit]:
        lines.append(f"  p={i}: gpu={gpu[i]!r} oracle={orc['fitness'][i]!r} E={orc['bound'][i]:.3g} "
                     f"flags={orc['flags'][i]}")
    return "\n".join(lines)
