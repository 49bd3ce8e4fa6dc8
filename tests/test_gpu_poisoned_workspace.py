"""Every kernel family on a workspace that starts out as NaN bit patterns, between guard bands.

compute-sanitizer is closed on the pool this repository is built on (profiles/r03_sanitizers.md), so its memcheck and
initcheck questions are put with means of our own: the caller-owned workspace of nh_init_lattice (include/nh.h) is cut
out of a larger buffer filled with 0xFF bytes -- NaN in FP32 and FP64 -- with 1 MiB of the same pattern on either side.
  - A kernel that writes outside the workspace (within 1 MiB) changes a guard byte.
  - A kernel that reads workspace memory nothing has written yet, or memory outside it, and lets the value reach a
    result, produces a NaN: every field that comes back must be finite (and |n| = 1).
What this cannot see: accesses that stray from one array of the workspace into its neighbour, and shared-memory races
(the bit-identity tests across launch shapes in test_gpu_parity.py are the evidence there).
The cases are those of tests/sanitizer_cases.py: one small run per kernel family.
"""
import pytest

from sanitizer_cases import lattice_cases, run

pytestmark = pytest.mark.gpu

GUARD = 1 << 20


def nh():
    import paper_2503_06610_b200 as m
    from paper_2503_06610_b200 import build
    build.build()
    return m


def test_poisoned_workspace_and_guard_bands():
    import torch
    m = nh()
    torch.cuda.set_stream(torch.cuda.Stream())      # (graph replay cannot capture the legacy default stream)
    held = []

    def make(**kw):
        nbytes = m.workspace_bytes(m.make_params(**kw))
        buf = torch.full((GUARD + nbytes + GUARD + 256,), 0xFF, dtype=torch.uint8, device="cuda")
        off = GUARD + (-(buf.data_ptr() + GUARD)) % 256
        held.append((buf, off, nbytes))
        return m.Lattice(workspace=buf[off:off + nbytes], **kw)

    try:
        for label, shape, precision, steps, options, knobs, params in lattice_cases(m):
            lat = run(m, label, shape, precision, steps, options, knobs, make=make, **params)      # asserts finite fields
            lat.synchronize()
            lat.close()
            buf, off, nbytes = held.pop()
            assert bool((buf[:off] == 0xFF).all()), "a write below the workspace: " + label
            assert bool((buf[off + nbytes:] == 0xFF).all()), "a write above the workspace: " + label
    finally:
        torch.cuda.set_stream(torch.cuda.default_stream())
