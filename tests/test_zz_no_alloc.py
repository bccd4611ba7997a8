"""nbs_blocks_x_static (include/nbs.h): eq. 4.1 through the entry point that allocates no device memory -- the staged
block rows live in the library's `static __device__` scratch array -- against nbs_blocks_x, which takes them from the
stream-ordered allocator.  Same kernels, so the results must agree within the parity bar of the other tests (they
are in fact bit-identical).  Collected last (file name): a failure here hides no other test under `pytest -x`.
"""
import numpy as np
import pytest

from paper_1604_07983_b200 import synth

pytestmark = pytest.mark.gpu

RTOL = 1e-10


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("no CUDA device: the gpu-marked tests need a B200")
    return torch


@pytest.fixture(scope="module")
def nbs():
    from paper_1604_07983_b200 import nbs as m
    return m


def load(torch, ctx, L, seed):
    S = [torch.from_numpy(synth.propagator(seed, i, 0, L, m)).cuda() for i, m in enumerate((0.20, 0.21, 0.30))]
    ctx.load(0, *S)
    return S  # borrowed by the library: keep alive


def assert_close(torch, got, ref, what):
    scale = ref.abs().max().item()
    assert scale > 0, what
    assert torch.isfinite(got.real).all() and torch.isfinite(got.imag).all(), what
    assert (got - ref).abs().max().item() <= RTOL * scale, what


def test_static_scratch_equals_allocating_path_two_calls_in_a_row(torch_cuda, nbs, oracle):
    """Every call shares one scratch array that keeps the last call's contents: alternate antisymmetric (compact rows)
    and full blocks so that each call finds the rows of another baryon, of another layout, in it; twice per baryon."""
    torch = torch_cuda
    L = 4
    with nbs.Nbs(L, 1, [("p", "n", "p", "n")]) as ctx:
        keep = load(torch, ctx, L, seed=31)
        out = torch.empty((L ** 3, 4, 12, 12, 12), dtype=torch.complex128, device="cuda")
        free_before = None
        for name in ["p", "L", "Xm", "S0", "p", "Xs", "Sm", "Xu", "n"]:
            ref = ctx.blocks_x(0, name)
            for call in range(2):
                out.fill_(complex(float("nan"), float("nan")))
                ctx.blocks_x_static(0, name, out)
                torch.cuda.synchronize()
                assert_close(torch, out, ref, (name, call))
                assert torch.equal(out.real, ref.real) and torch.equal(out.imag, ref.imag), (name, call)
                if free_before is None:  # after the first call: kernels loaded, scratch address looked up
                    free_before = torch.cuda.mem_get_info()[0]
        # no device memory was taken by the later calls (the output tensor is reused)
        assert torch.cuda.mem_get_info()[0] >= free_before
        del keep
    # grounded in the oracle as well, at the size the oracle's blocks take no time
    L = 2
    S = {f: synth.propagator(5, i, 0, L, m) for i, (f, m) in enumerate(zip("uds", (0.20, 0.21, 0.30)))}
    with nbs.Nbs(L, 1, [("p", "n", "p", "n")]) as ctx:
        dev = {f: torch.from_numpy(S[f]).cuda() for f in "uds"}
        ctx.load(0, dev["u"], dev["d"], dev["s"])
        out = torch.empty((L ** 3, 4, 12, 12, 12), dtype=torch.complex128, device="cuda")
        for name in oracle.BARYONS:
            for call in range(2):
                got = ctx.blocks_x_static(0, name, out).cpu().numpy()
                ref = oracle.block(S, name)
                assert np.abs(got - ref).max() <= RTOL * np.abs(ref).max(), (name, call)


def test_static_scratch_limit_and_sharing_between_contexts(torch_cuda, nbs):
    """Up to the stated maximum (32 MiB of staged rows: a full block at 6^3, a compact one at 8^3) the entry point
    works, beyond it it refuses with the sizes in the message and launches nothing; two contexts share the array."""
    torch = torch_cuda
    assert nbs.STATIC_SCRATCH_BYTES == 32 << 20
    with nbs.Nbs(6, 1, [("p", "n", "p", "n")]) as c6, nbs.Nbs(8, 1, [("p", "n", "p", "n")]) as c8:
        k6 = load(torch, c6, 6, seed=32)
        k8 = load(torch, c8, 8, seed=33)
        o6 = torch.empty((6 ** 3, 4, 12, 12, 12), dtype=torch.complex128, device="cuda")
        o8 = torch.empty((8 ** 3, 4, 12, 12, 12), dtype=torch.complex128, device="cuda")
        assert 6 ** 3 * 6960 * 16 <= nbs.STATIC_SCRATCH_BYTES < 8 ** 3 * 6960 * 16
        assert 8 ** 3 * 3472 * 16 <= nbs.STATIC_SCRATCH_BYTES
        for call in range(2):  # the two contexts take turns on the same array (one stream: ordered)
            c6.blocks_x_static(0, "L", o6)
            c8.blocks_x_static(0, "Sp", o8)
            torch.cuda.synchronize()
            assert_close(torch, o6, c6.blocks_x(0, "L"), ("L", call))
            assert_close(torch, o8, c8.blocks_x(0, "Sp"), ("Sp", call))
        launches = c8.kernel_launches()
        o8.fill_(7.0)
        with pytest.raises(nbs.NbsError) as ei:
            c8.blocks_x_static(0, "L", o8)  # 57 016 320 bytes of staged rows
        assert ei.value.code == nbs.NBS_EINVAL
        assert "57016320" in str(ei.value) and str(32 << 20) in str(ei.value)
        torch.cuda.synchronize()
        assert c8.kernel_launches() == launches and bool((o8 == 7.0).all())
        # the context stays usable after the refusal
        c8.blocks_x_static(0, "Xm", o8)
        torch.cuda.synchronize()
        assert_close(torch, o8, c8.blocks_x(0, "Xm"), "Xm")
        del k6, k8
