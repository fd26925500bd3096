"""Small seeded models for the oracle pins (numpy only; no likelihood arithmetic here)."""
import numpy as np


def random_model(oracle, seed, R, H, C, n_data, n_mc, weighted=True):
    rs = np.random.RandomState(seed)
    res_chan = (np.arange(R) % C).astype(np.int32)

    def sample(n, w):
        mass = rs.uniform(0.3, 3.0, size=(C, n))
        amp = rs.normal(size=(R, H, n, 2))
        return oracle.Sample(mass, amp, rs.uniform(0.5, 1.5, size=n) if w else None)

    return oracle.Model(res_chan, sample(n_data, weighted), sample(n_mc, False))


def random_theta(seed, R):
    rs = np.random.RandomState(seed)
    th = np.empty((R, 4))
    th[:, 0] = rs.uniform(0.5, 1.5, R)
    th[:, 1] = rs.uniform(-np.pi, np.pi, R)
    th[:, 2] = rs.uniform(0.5, 2.8, R)
    th[:, 3] = rs.uniform(0.05, 0.4, R)
    return th.reshape(-1)


def rel_l2(a, b):
    a = np.asarray(a, dtype=np.longdouble)
    b = np.asarray(b, dtype=np.longdouble)
    return float(np.sqrt(((a - b) ** 2).sum()) / np.sqrt((b ** 2).sum()))
