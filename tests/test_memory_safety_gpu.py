"""Memory-safety checks of every kernel (-m gpu), standing in for compute-sanitizer, which is closed on this GPU
pool (profiles/r2_sanitizer_closed.md).

The bindings allocate their outputs, workspaces and preconditioner buffers with ``torch.empty``.  Here that call
is replaced, inside the binding modules only, by an allocator that puts every buffer between two guard bands
filled with a pattern and fills the buffer itself with 0xFF bytes (NaN as float64 / float32, -1 as int64):

* a kernel that writes outside a buffer it was given damages a guard band        -> checked after every case;
* a kernel that reads workspace or output memory before writing it produces NaN  -> every case checks its
  results to be finite, and the solves check their residuals;
* a result that depends on stale memory or on the timing of a race differs from run to run -> the reproducible
  paths are run repeatedly, with different poison, and compared bit for bit.

The cases are those of tests/kernel_cases.py: every kernel of the library, every code path.
"""
import contextlib

import numpy as np
import pytest
import torch

import kernel_cases
from paper_1602_02170_b200 import binding, rigid, workloads

pytestmark = pytest.mark.gpu

GUARD = 4096          # bytes on each side; a multiple of the 256-byte alignment the library asks for
PATTERN = 0xA5


class GuardedTorch:
    """Stands in for the ``torch`` module inside the bindings: ``empty`` returns guarded, poisoned CUDA buffers."""

    def __init__(self, poison: int = 0xFF):
        self.poison = poison
        self.buffers = []

    def __getattr__(self, name):
        return getattr(torch, name)

    def empty(self, *size, dtype=torch.float32, device=None, **kw):
        if len(size) == 1 and isinstance(size[0], (tuple, list, torch.Size)):
            size = tuple(size[0])
        dev = torch.device(device) if device is not None else torch.device("cpu")
        if dev.type != "cuda" or kw.get("pin_memory"):
            return torch.empty(*size, dtype=dtype, device=device, **kw)
        n = int(np.prod(size)) if len(size) else 1
        nbytes = n * torch.empty(0, dtype=dtype).element_size()
        padded = (nbytes + 255) // 256 * 256
        raw = torch.empty(2 * GUARD + padded, dtype=torch.uint8, device=dev)
        raw.fill_(PATTERN)
        raw[GUARD:GUARD + nbytes].fill_(self.poison)
        self.buffers.append((raw, nbytes))
        return raw[GUARD:GUARD + nbytes].view(dtype).view(size)

    def check(self):
        torch.cuda.synchronize()
        for raw, nbytes in self.buffers:
            lo, hi = raw[:GUARD], raw[GUARD + nbytes:]
            assert bool((lo == PATTERN).all()), f"write BELOW a buffer of {nbytes} bytes"
            assert bool((hi == PATTERN).all()), f"write ABOVE a buffer of {nbytes} bytes"
        return len(self.buffers)


@contextlib.contextmanager
def guarded(poison=0xFF):
    g = GuardedTorch(poison)
    saved = binding.torch, rigid.torch
    binding.torch = rigid.torch = g
    try:
        yield g
    finally:
        binding.torch, rigid.torch = saved


@pytest.mark.parametrize("name", list(kernel_cases.CASES))
def test_no_write_outside_a_buffer_and_no_read_before_write(name):
    with guarded() as g:
        kernel_cases.CASES[name]()
        n = g.check()
    assert n > 0                                   # the instrumentation saw the bindings' allocations
    print(f"{name}: {n} guarded buffers intact")


def test_guard_bands_do_catch_an_overrun():
    """The instrument itself: a workspace that is too short by one row of partial sums must trip a guard --
    reached by handing the library a correctly sized view of a deliberately undersized guarded region."""
    g = GuardedTorch()
    t = g.empty(1000, dtype=torch.float64, device="cuda")
    raw, _ = g.buffers[0]
    raw[GUARD + 8000: GUARD + 8008].fill_(0)       # what an off-by-one store would do
    with pytest.raises(AssertionError):
        g.check()
    assert bool(torch.isnan(t).all())              # and the poison reads back as NaN


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_reproducible_paths_are_bit_identical_whatever_was_in_the_workspace(prec):
    """Plain kernel (k = 2; row range), preconditioner build + application and the GMRES solve with the plain
    product: bit-identical across runs whose workspaces start as NaN, as zeros and as the previous run's
    leftovers.  A race on the shared-memory staging, or a read of stale workspace, would show here."""
    dt = torch.float64 if prec == "f64" else torch.float32
    w = workloads.config2(seed=7, n_bodies=70, k=2)            # 1,050 blobs (< 1,152): the plain kernel also inside the solve
    hb = workloads.bodies_of(w)
    pos, lam = torch.from_numpy(w.pos).to(dt).cuda(), torch.from_numpy(w.force).to(dt).cuda()
    pos64 = torch.from_numpy(w.pos).cuda()
    ref = None
    for rep, poison in enumerate((0xFF, 0x00, 0x7F, 0xFF)):
        with guarded(poison) as g:
            u = binding.rpy_wall_matvec(pos, lam)
            ur = binding.rpy_free_matvec(pos, lam, rows=(100, 900))
            db = rigid.bodies(pos64, torch.from_numpy(hb.q).cuda(), hb.offsets)
            pc = rigid.rpy_rigid_precond_build(db, "wall")
            x = torch.arange(db.n, dtype=torch.float64, device="cuda").sin()
            z = rigid.rpy_rigid_precond_apply(pc, x)
            r = rigid.rpy_rigid_mobility_solve(db, pc, torch.from_numpy(hb.F).cuda(), None, "wall", tol=1e-9,
                                               matvec_prec=prec if prec == "f64" else "mixed")
            g.check()
        got = (u.clone(), ur.clone(), z.clone(), r["U"].clone(), r["lambda"].clone(), r["n_iter"])
        if ref is None:
            ref = got
        else:
            for a, b in zip(ref[:-1], got[:-1]):
                assert torch.equal(a, b), f"run {rep} differs"
            assert ref[-1] == got[-1]


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_symmetric_kernel_is_reproducible_to_rounding_under_poison(prec):
    """The symmetric kernel's transposed half lands with fp64 atomics: reproducible to rounding of the double
    sums, and independent of what the accumulator slice held before (the prepack kernel clears it)."""
    dt = torch.float64 if prec == "f64" else torch.float32
    w = workloads.config2(seed=8, n_bodies=400)                # 6,000 blobs
    pos, lam = torch.from_numpy(w.pos).to(dt).cuda(), torch.from_numpy(w.force).to(dt).cuda()
    outs = []
    for poison in (0xFF, 0x00, 0x3C):
        with guarded(poison) as g:
            outs.append(binding.rpy_wall_matvec(pos, lam).double())
            g.check()
    for o in outs[1:]:
        assert float((o - outs[0]).norm() / outs[0].norm()) <= 1e-14
