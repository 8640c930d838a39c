"""The parity harness's own NumPy restatement of the collapse criterion (Eq. 18, reading A17)
agrees with the oracle's orc_collapse_test on perturbed tower states."""
import numpy as np

from paper_2606_28394_b200 import workloads as W
from test_gpu_parity import collapse_flags


def test_collapse_flags_match_oracle(orc):
    wl = W.make_config(2, n_envs=8)
    B = wl.params.n_bodies
    rng = np.random.default_rng(5)
    st = wl.state.copy()
    st[:, 0:3, :B] += rng.normal(0, 0.03, (8, 3, B)).astype(np.float32)
    q = st[:, 3:7, :B] + rng.normal(0, 0.2, (8, 4, B)).astype(np.float32)
    st[:, 3:7, :B] = q / np.linalg.norm(q, axis=1, keepdims=True)
    st[:, 7:13, :B] = rng.normal(0, 0.05, (8, 6, B)).astype(np.float32)
    st[4:, 7:13, :] = 0                      # at rest: kinetic-energy condition fails
    st[2, 0:3, :] = wl.state[2, 0:3, :]      # not displaced: displacement condition fails
    got = collapse_flags(st, wl.state, wl.props, B)
    bod = orc.unpack_tiles(st, wl.props, B); b0 = orc.unpack_tiles(wl.state, wl.props, B)
    ref = [orc.collapse_test(bod, b0.x[e], b0.q[e], e=e)[0] for e in range(8)]
    assert got.tolist() == ref and any(ref) and not all(ref)
