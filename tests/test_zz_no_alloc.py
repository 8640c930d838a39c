"""jenga_narrowphase_static: the narrowphase for callers that cannot give the library scratch memory.

Some users of libjenga.so cannot allocate device memory at the moment they need contacts: their host program handed out
all of its GPU memory at start-up, or they run inside a loop where the stall of a cudaMalloc is not acceptable, or they
are in a region where the allocator must not be called.  The ordinary path needs a caller-allocated, zero-filled
jenga_buffers.scratch before a world can even be created; this entry point works in an 8 MiB array that is part of the
library image instead (include/jenga.h).  What a user has to know, and what is checked here:

  * same result as jenga_narrowphase on the same inputs (the test asks for the same bits, which is inside the 1e-6 m /
    1e-4 rad tolerance the parity tests use), on consecutive calls of different sizes: the shared array keeps the previous
    call's contents and they must not matter;
  * free device memory is the same before and after a call (nothing was allocated or freed);
  * a batch beyond the array is refused with E_STATIC_CAPACITY before anything is launched.

The file name sorts last on purpose: the suite runs with `pytest -x`, and a failure here must not hide the parity tests.
It passes alone in a fresh process (the first call then does the per-device set-up) and after the other tests.
"""
import ctypes as C

import numpy as np
import pytest

from paper_2606_28394_b200 import workloads as W


def _existing_path(J, wl, warm_steps):
    """Contacts of the existing path (world with caller scratch): a few steps to get a lived-in state, then S2 + S3."""
    import torch
    world = J.World(wl.params, wl.state, wl.props, wl.mu)
    if warm_steps:
        world.step(warm_steps)
    world.broadphase()
    world.status.zero_()                       # only what the narrowphase reports is compared
    world.narrowphase(); torch.cuda.synchronize()
    return world


def _static_path(J, world):
    """The same inputs (state, props, pairs, n_pairs of `world`) through the entry point that allocates nothing.
    The output tensors are made here, by the caller, before the call; they start as a sentinel."""
    import torch
    contacts = torch.full_like(world.contacts, -7.0)
    n_contacts = torch.full_like(world.n_contacts, -7)
    status = torch.zeros_like(world.status)
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info(world.dev)[0]
    J.jenga_narrowphase_static(world.desc, world.state, world.props, world.pairs, world.n_pairs, contacts, n_contacts, status)
    torch.cuda.synchronize()
    free1 = torch.cuda.mem_get_info(world.dev)[0]
    return contacts, n_contacts, status, free0, free1


def _same_contacts(world, contacts, n_contacts, status):
    import torch
    assert torch.equal(n_contacts, world.n_contacts)
    assert torch.equal(status, world.status)
    total = 0
    for e in range(world.wp.n_envs):
        n = int(n_contacts[e].item())
        total += n
        # the very same words: normals, depths, points and the (pair position, slot, axis) tags
        assert torch.equal(contacts[e, :n].view(torch.int32), world.contacts[e, :n].view(torch.int32)), f"env {e}"
        assert bool((contacts[e, n:] == -7.0).all()), f"env {e}: wrote beyond its contact count"
    return total


@pytest.mark.gpu
def test_static_narrowphase_equals_existing_path_on_consecutive_calls():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    from paper_2606_28394_b200 import binding as J
    J.lib()
    # call 1: tumbling debris (every manifold kind: face, edge, ground); call 2: towers with a different env count, so the
    # per-env regions of the shared array fall elsewhere and hold call 1's leftovers; call 3: call 1's inputs once more
    debris = _existing_path(J, W.make_config(3, n_envs=7), 150)
    towers = _existing_path(J, W.make_config(2, n_envs=10), 25)
    tall = _existing_path(J, W.make_config(4, n_envs=3), 10)          # 90 bodies: other max_contacts, other region size
    totals, frees = [], []
    for k, world in enumerate((debris, towers, debris, tall)):
        contacts, n_contacts, status, free0, free1 = _static_path(J, world)
        totals.append(_same_contacts(world, contacts, n_contacts, status))
        frees.append((k, free0, free1))
    assert min(totals) > 100, totals                                  # the comparison was not empty
    assert totals[0] == totals[2]
    # calls after the first (set-up done): free device memory unchanged across the call
    for k, free0, free1 in frees[1:]:
        assert free0 == free1, f"call {k}: free device memory changed by {free0 - free1} bytes"
    for w in (debris, towers, tall):
        w.destroy()


def test_static_narrowphase_limit_is_checked_before_any_launch():
    """No GPU needed: sizes are validated on the host first.  8 MiB / 15,616 B = 537 envs of 54 blocks."""
    from paper_2606_28394_b200 import binding as J
    L = J.lib()
    wp = W.make_config(2, n_envs=2).params
    d = J.make_desc(wp)
    per_env = J.jenga_narrowphase_static_env_bytes(d)
    assert per_env == 4 * 64 * -(-(16 + 22 * (wp.max_contacts // 4)) // 64) == 15616 and per_env % 256 == 0
    fits = J.STATIC_SCRATCH_BYTES // per_env
    assert fits == 537
    dummy = C.c_void_p(256)                                           # aligned, never dereferenced: the call stops earlier
    args = [dummy] * 7 + [None]
    d.n_envs = fits + 1
    assert L.jenga_narrowphase_static(C.byref(d), *args) == J.E_STATIC_CAPACITY
    assert b"built-in" in L.jenga_strerror(J.E_STATIC_CAPACITY) and b"8 MiB" in L.jenga_strerror(J.E_STATIC_CAPACITY)
    d.n_envs = 1 << 30                                                # no overflow in the size product
    assert L.jenga_narrowphase_static(C.byref(d), *args) == J.E_STATIC_CAPACITY
    bad = J.make_desc(wp); bad.max_contacts = 6
    assert L.jenga_narrowphase_static(C.byref(bad), *args) == -1 and J.jenga_narrowphase_static_env_bytes(bad) == 0
    ok = J.make_desc(wp)
    assert L.jenga_narrowphase_static(C.byref(ok), None, *args[1:]) == -1          # NULL input
