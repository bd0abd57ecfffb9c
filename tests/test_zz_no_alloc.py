"""pinsage_head_static: the head for callers that must not allocate (CUDA graph capture, serving loops).

Its scratch is a file-scope __device__ array of the library (gemm_head.cu) instead of the context's
cudaMalloc'ed buffer.  Checked here: same bits as the existing path (pinsage_head, which runs the same
kernel on allocated scratch; the tolerance the head tests use against the oracle holds for it there) on two
calls in a row that leave different contents in the shared array, no change in the device's free memory
across the calls, and a clear rejection beyond the limits.  Collected last on purpose (file name)."""
import pytest
import torch

from paper_1806_01973_b200 import binding

pytestmark = pytest.mark.gpu
DEV = "cuda:0"


def _case(M, d, g1, d_out, seed):
    g = torch.Generator().manual_seed(seed)
    h = torch.randn((M, d), generator=g).to(torch.bfloat16).to(DEV)
    head = {"G1": (torch.randn((g1, d), generator=g) * d ** -0.5).to(torch.bfloat16).to(DEV),
            "g": (torch.randn((g1,), generator=g) * 0.05).to(DEV),
            "G2": (torch.randn((d_out, g1), generator=g) * g1 ** -0.5).to(torch.bfloat16).to(DEV)}
    return h, head


def test_head_static_matches_the_allocating_path_twice_and_allocates_nothing():
    cases = [_case(50_011, 256, 256, 256, 70),      # CTA pairs, every scratch slot of every CTA in use
             _case(20_000, 256, 128, 64, 71),       # narrower a tiles over the first call's leftovers
             _case(130, 136, 72, 40, 72)]           # too few tiles for pairs: the single-CTA form
    with binding.Context(0) as ref_ctx, binding.Context(0) as ctx:
        refs = [ref_ctx.pinsage_head(h, head) for h, head in cases]
        outs = [torch.full_like(r, float("nan")) for r in refs]
        # set-up: the first call on a device resolves the array's address and loads the kernels
        ctx.pinsage_head_static(cases[0][0], cases[0][1], outs[0])
        torch.cuda.synchronize()
        outs[0].fill_(float("nan"))
        again = torch.full_like(refs[0], float("nan"))
        torch.cuda.synchronize()
        free0 = torch.cuda.mem_get_info(0)[0]
        l0 = ctx.pinsage_launch_count()
        for (h, head), out in zip(cases, outs):     # calls in a row on one stream, no sync in between
            ctx.pinsage_head_static(h, head, out)
        ctx.pinsage_head_static(cases[0][0], cases[0][1], again)
        torch.cuda.synchronize()
        assert ctx.pinsage_launch_count() - l0 == 4          # one launch per call
        assert torch.cuda.mem_get_info(0)[0] == free0, "pinsage_head_static changed the device's free memory"
        for out, ref in zip(outs + [again], refs + [refs[0]]):
            assert torch.isfinite(out.float()).all()
            assert torch.equal(out.view(torch.int16), ref.view(torch.int16))
            err = (out.double() - ref.double()).norm(dim=1) / ref.double().norm(dim=1).clamp_min(1e-30)
            assert float(err.max()) <= 1e-2          # (the bf16 tolerance of the parity tests; 0 here)


def test_head_static_rejects_what_the_static_array_cannot_hold():
    with binding.Context(0) as ctx:
        for (M, d, g1, d_out), dtype in (((1000, 256, 512, 256), torch.bfloat16),     # g1 beyond the array's rows
                                         ((1000, 256, 256, 512), torch.bfloat16),
                                         ((1000, 64, 64, 32), torch.float32)):
            h, head = _case(M, d, g1, d_out, 73)
            h = h.to(dtype)
            head = {k: (v if k == "g" else v.to(dtype)) for k, v in head.items()}
            out = torch.zeros((M, d_out), dtype=dtype, device=DEV)
            l0 = ctx.pinsage_launch_count()
            with pytest.raises(binding.PinsageError) as ex:
                ctx.pinsage_head_static(h, head, out)
            assert "pinsage_head_static" in str(ex.value)
            assert ctx.pinsage_launch_count() == l0 and not out.any()
