"""Next row (GNN part): the INT8 GNN on the tensor cores (ETX_PREC_INT8, tcgen05.mma.kind::i8) vs the
quantised oracle.  Every integer code is reproducible, and all float steps are single rounded fp32 operations, so the
final encodings h, e must be BIT-EQUAL to the oracle's; the scores differ only by the sigmoid's exp (fp32 vs double)."""
import numpy as np
import pytest
import torch

from conftest import layout_dict, oracle_path
from oracle import etx_oracle as orc
from paper_2508_07423_b200 import synth

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2508_07423_b200 import binding, build
    build.build()
    return binding


def gpu_int8(B, cfg, batch, blob, ora, alpha):
    etx = B.Etx(B.make_desc(cfg, precision=synth.PREC_INT8), blob)
    etx.etx_set_int8_ranges(alpha)
    dev = etx.device
    db = B.DeviceBatch(batch, dev)
    cap = len(ora["src"]) + 5
    etx.ensure_workspace(db.n_events, db.n_hits, cap)
    g = B.DeviceGraph(db.n_hits, cap, dev)
    E = etx.etx_build_graph(db, torch.from_numpy(ora["emb"]).to(dev), synth.r2_max(cfg), cfg.max_plane_gap, g)
    assert E == len(ora["src"])
    e = torch.empty(max(E, 1), cfg.gnn_hidden, device=dev)
    h = torch.empty(db.n_hits, cfg.gnn_hidden, device=dev)
    s = torch.empty(max(E, 1), device=dev)
    etx.etx_gnn_forward(db, g, e, h)
    etx.etx_edge_scores(g, e, s)
    torch.cuda.synchronize()
    assert etx.launch_count() > 0
    return h.cpu().numpy(), e[:E].cpu().numpy(), s[:E].cpu().numpy()


def check(B, cfg, batch, blob, ora, alpha):
    lay = layout_dict(cfg)
    h0, e0, logit0, s0 = orc.gnn_forward_int8(ora["f_node"], ora["src"], ora["dst"], cfg.n_iter, blob, lay, alpha)
    h, e, s = gpu_int8(B, cfg, batch, blob, ora, alpha)
    nh, ne = int((h != h0).sum()), int((e != e0).sum())
    print(f"{cfg.name}: N={len(h0)} E={len(e0)}  h mismatches {nh}, e mismatches {ne}, max |score - int8 oracle| = "
          f"{np.abs(s.astype(np.float64) - s0).max():.3g}; int8 vs FP32 oracle: max {np.abs(s.astype(np.float64) - ora['scores']).max():.3g}, "
          f"median {np.median(np.abs(s.astype(np.float64) - ora['scores'])):.3g}")
    np.testing.assert_array_equal(h, h0)
    np.testing.assert_array_equal(e, e0)
    np.testing.assert_allclose(s, s0, rtol=0, atol=1e-6)
    return s


def test_int8_gnn_c1_bit_equal(B, c1, c1_oracle):
    cfg, batch, blob = c1
    s = check(B, cfg, batch, blob, c1_oracle, synth.int8_gnn_alpha(cfg))
    assert np.abs(s.astype(np.float64) - c1_oracle["scores"]).max() < 0.25      # a quantised model, not a broken one


def test_int8_gnn_multi_event_ragged_and_clipping(B):
    cfg = synth.CONFIGS["c2"]
    batch = synth.generate_events(cfg, range(500, 505))            # 5 events: several tiles, ragged tails, hits != edges
    blob = synth.generate_weights(cfg)
    ora = oracle_path(cfg, batch, blob)
    al = synth.int8_gnn_alpha(cfg)
    check(B, cfg, batch, blob, ora, al)
    narrow = {k: [0.25 * a for a in v] for k, v in al.items()}      # ranges 4x too narrow: the clip of Eq. 4.33 is exercised
    check(B, cfg, batch, blob, ora, narrow)


def test_int8_needs_ranges(B, c1, c1_oracle):
    cfg, batch, blob = c1
    etx = B.Etx(B.make_desc(cfg, precision=synth.PREC_INT8), blob)
    db = B.DeviceBatch(batch, etx.device)
    cap = len(c1_oracle["src"]) + 5
    etx.ensure_workspace(1, db.n_hits, cap)
    g = B.DeviceGraph(db.n_hits, cap, etx.device)
    etx.etx_build_graph(db, torch.from_numpy(c1_oracle["emb"]).to(etx.device), synth.r2_max(cfg), cfg.max_plane_gap, g)
    with pytest.raises(B.EtxError) as ei:
        etx.etx_gnn_forward(db, g, torch.empty(cap, cfg.gnn_hidden, device=etx.device))
    assert ei.value.status == B.ETX_ERR_INVALID
    with pytest.raises(B.EtxError) as ei:
        etx.etx_set_int8_ranges({k: [-1.0] * 3 for k in synth.int8_gnn_alpha(cfg)})
    assert ei.value.status == B.ETX_ERR_INVALID
