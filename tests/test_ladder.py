"""Host-side ladder arithmetic (temperatures "chosen such that the acceptance rate of swaps is independent
of the temperatures") and the paper's workload families.  CPU only; no compute calls."""
import numpy as np

from paper_1211_0780_b200 import inputs, ladder


def test_paper_families_match_the_paper():
    """34 temperatures in [2.1, 2.3] for L = 64, 80, 96, 128; 13 in [2.19, 2.21] for L = 160."""
    fam = {f.L: f for f in inputs.PAPER_FAMILIES}
    assert sorted(fam) == [64, 80, 96, 128, 160]
    for L in (64, 80, 96, 128):
        assert fam[L].R == 34 and (fam[L].T_lo, fam[L].T_hi) == (2.1, 2.3)
    assert fam[160].R == 13 and (fam[160].T_lo, fam[160].T_hi) == (2.19, 2.21)
    for f in inputs.PAPER_FAMILIES:
        b = inputs.betas_of_family(f)
        assert b.shape == (f.R,) and b[0] == 1.0 / f.T_hi and b[-1] == 1.0 / f.T_lo
        assert np.all(np.diff(b) > 0)
        assert np.allclose(b[1:] / b[:-1], (b[-1] / b[0]) ** (1.0 / (f.R - 1)), rtol=1e-12)     # geometric: NOT uniform in beta
        assert np.diff(b).max() / np.diff(b).min() > 1.005
        assert b[0] < 1.0 / 2.2019 < b[-1]                                                       # T_c of P:76 is inside
        assert inputs.paper_family(f.name) is f


def test_respace_keeps_the_ends_and_moves_spacings_towards_flat_acceptance():
    b = inputs.geometric_beta_ladder(2.1, 2.3, 12)
    flat = np.full(11, 0.8)
    assert np.allclose(ladder.respace(b, flat), b, rtol=0, atol=1e-15), "flat acceptance is a fixed point"
    a = np.linspace(0.95, 0.55, 11)                      # the cold end rejects more: its spacings must shrink
    nb = ladder.respace(b, a)
    assert nb[0] == b[0] and nb[-1] == b[-1] and np.all(np.diff(nb) > 0)
    ratio = np.diff(nb) / np.diff(b)
    assert np.all(np.diff(ratio) < 0) and ratio[0] > 1 > ratio[-1]
    # a model system with rejection = c_k * spacing converges to flat rejection
    c = np.linspace(1.0, 3.0, 11) * 40.0
    x = b.copy()
    for _ in range(40):
        x = ladder.respace(x, 1.0 - c * np.diff(x), gamma=0.5)
    rej = c * np.diff(x)
    assert rej.std() / rej.mean() < 1e-3 and x[0] == b[0] and abs(x[-1] - b[-1]) < 1e-15
    assert np.array_equal(ladder.respace(b[:2], [0.5]), b[:2])


class _FakeXY:
    """Stands in for binding.XY: pair k accepts a fixed fraction of its attempts (pairs with k = n_pt mod 2)."""
    def __init__(self, R, frac):
        self.R, self.frac, self.n_pt = R, np.asarray(frac), 0
        self.acc = np.zeros(R - 1)

    def get_accept_counts(self):
        return None, self.acc.copy()

    def get_counters(self):
        return np.array([self.n_pt, self.n_pt, self.n_pt], dtype=np.uint32)

    def mcs(self, n):
        for _ in range(n):
            k = np.arange(self.n_pt & 1, self.R - 1, 2)
            self.acc[k] += self.frac[k]
            self.n_pt += 1


def test_measured_acceptance_counts_the_attempts_of_each_pair():
    frac = np.array([0.9, 0.5, 0.7, 0.2, 1.0])
    for start, n in ((0, 10), (1, 10), (0, 7), (3, 5)):
        xy = _FakeXY(6, frac)
        xy.mcs(start)
        a = ladder.measure_swap_acceptance(xy, n)
        assert np.allclose(a, frac), (start, n, a)
