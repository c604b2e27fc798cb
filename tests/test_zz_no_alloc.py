"""-m gpu test of protokv_query_attention_static (include/protokv.h; csrc/static_scratch.cu): the attention of Alg. 4
 with its split-context partials in the library's file-scope device array, for callers that may not
allocate.  Checked against the existing entry point (protokv_query_attention_ex, partials in the workspace, whatever
route the state takes by default) within the tolerance the route-agreement tests use, on two calls in a row.

The file name sorts last on purpose: the suite runs with pytest -x, so a failure here hides no other test."""
import pytest
import torch

import gen
from gpu_helpers import make_gpu
from paper_2606_26762_b200 import binding as B

pytestmark = pytest.mark.gpu

ATOL, RTOL = 1e-2, 2e-2          # tests/test_gpu_alloc.py::test_ragged_attention_routes_agree


def _stream(spec, gpu, frames):
    s = gen.grid_positions(spec, device="cuda")
    for f in range(frames):
        K, V = gen.frame_kv(spec, f, device="cuda")
        gpu.append_frame(K, V, s)


@pytest.mark.parametrize("name,frames,flags", [("c2", 30, 0), ("c1", 24, 0), ("c2", 24, B.ROPE)])
def test_static_scratch_attention_matches_the_workspace_path_twice(name, frames, flags):
    spec = gen.spec_for(name, n_frames=frames)
    gpu = make_gpu(spec, flags=flags)
    assert gpu.static_scratch_bytes == 8 << 20
    _stream(spec, gpu, frames)
    Qa = gen.queries(spec, 0).cuda()[:, :, :1].contiguous()             # one-token query (decode-style)
    Qb = gen.queries(spec, 1).cuda()                                    # the configured multi-token query
    ref_a = gpu.query_attention_ex(Qa, n_q=1).float()
    ref_b, lse_ref = gpu.query_attention_ex(Qb, return_lse=True, run_synthesis=False)
    out_a, out_b = torch.empty_like(Qa), torch.empty_like(Qb)
    lse_b = torch.empty_like(lse_ref)
    torch.cuda.synchronize()
    # two calls in a row, different shapes: the second finds the first one's partials in the array
    gpu.query_attention_static(Qa, out_a, n_q=1, run_synthesis=False)
    free0 = torch.cuda.mem_get_info()[0]
    gpu.query_attention_static(Qb, out_b, lse=lse_b, run_synthesis=False)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0                        # no device memory taken by the call
    assert torch.allclose(out_a.float(), ref_a, atol=ATOL, rtol=RTOL), (out_a.float() - ref_a).abs().max()
    assert torch.allclose(out_b.float(), ref_b.float(), atol=ATOL, rtol=RTOL), (out_b.float() - ref_b.float()).abs().max()
    assert torch.allclose(lse_b, lse_ref, atol=5e-3, rtol=0)
    # and again after the state has moved on (synthesis inside the call), same array
    _stream(spec, gpu, 2)
    gpu.query_attention_static(Qa, out_a, n_q=1)
    ref_a2 = gpu.query_attention_ex(Qa, n_q=1, run_synthesis=False).float()
    assert torch.allclose(out_a.float(), ref_a2, atol=ATOL, rtol=RTOL)
    assert not torch.equal(ref_a2, ref_a)
    assert gpu.error_flags() == 0
    gpu.close()


def test_static_scratch_rejects_what_does_not_fit_and_serves_the_c3_decode_query():
    """Config 3 (112 banks): the 32-token query needs 13 MB of partials per split -> PROTOKV_EUNSUPPORTED, state untouched;
    its one-token query (0.4 MB per split) runs in the launch configuration bench.py's decode query has."""
    spec = gen.spec_for("c3")
    gpu = make_gpu(spec)
    _stream(spec, gpu, spec.near_frames + 3)
    Q = gen.queries(spec, 0).cuda()
    out = torch.empty_like(Q)
    launches = gpu.kernel_launches
    with pytest.raises(B.ProtoKVError, match="static scratch holds 8388608"):
        gpu.query_attention_static(Q, out)
    assert gpu.kernel_launches == launches                              # nothing ran, not even the synthesis
    Q1 = Q[:, :, :1].contiguous()
    out1 = torch.empty_like(Q1)
    for _ in range(2):
        gpu.query_attention_static(Q1, out1, n_q=1)
    ref = gpu.query_attention_ex(Q1, n_q=1, run_synthesis=False).float()
    assert torch.allclose(out1.float(), ref, atol=ATOL, rtol=RTOL), (out1.float() - ref).abs().max()
    assert torch.isfinite(out1.float()).all() and out1.float().abs().max() > 0
    gpu.close()
