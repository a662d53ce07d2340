"""Reduced form of the paper's accuracy study (section 3.3, Eq. 22; paper_2306_04322_b200/accuracy.py): the ordering
the paper reports must come out of the GPU path -- FS most accurate, FS-FD O(dl^4) next, FS-FD O(dl^2) and FD last and
alike."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def test_error_ordering_of_the_variants():
    from paper_2306_04322_b200 import accuracy, pf, synth
    p, length, nr, n = 4, 200.0, 512, 128
    c0, eta0, _ = synth.init_b((nr, nr), p)
    c1, eta1, _, _ = accuracy.advance(pf, nr, p, length / nr, 5e-4, 1.0, c0, eta0)          # stand-in pre-evolution
    cr, er, _, _ = accuracy.advance(pf, nr, p, length / nr, 5e-4, 2.0, c1, eta1)            # reference, t = 1 .. 3
    r = nr // n
    ci, ei = np.ascontiguousarray(c1[::r, ::r]), np.ascontiguousarray(eta1[:, ::r, ::r])
    rc, rs = cr[::r, ::r], er.sum(0)[::r, ::r]
    err = {}
    for name, method, kind, dt in (("fs", "fs", 0, 1e-3), ("c4", "fs", 2, 1e-3), ("c2", "fs", 1, 1e-3), ("fd", "fd", 0, 1e-3)):
        gc, ge, _, _ = accuracy.advance(pf, n, p, length / n, dt, 2.0, ci, ei, method, kind)
        assert np.isfinite(gc).all() and np.isfinite(ge).all()
        err[name] = (accuracy.eq22_percent(gc, rc), accuracy.eq22_percent(ge.sum(0), rs))
    for k in (0, 1):                                       # E_c and E_eta
        assert err["fs"][k] < err["c4"][k] < err["c2"][k]
        assert 0.3 < err["fd"][k] / err["c2"][k] < 3.0     # same second-order stencil symbol, explicit vs semi-implicit in time
