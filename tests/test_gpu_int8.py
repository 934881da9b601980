"""Next row (embedding part): INT8 embedding MLP on the GPU vs the oracle (P:2723-2742,
Eqs. 4.31-4.33).  Floating point only decides integer codes through single rounded fp32 operations that both sides
perform identically, so the embeddings must be BIT-equal, and with them the graph built from them."""
import dataclasses

import numpy as np
import pytest
import torch

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


def oracle_int8(cfg, batch, blob, alphas):
    spec = synth.model_layout(cfg)[0]
    fe, _ = orc.features(batch, synth.NORM_CENTER, synth.NORM_SCALE)
    return orc.mlp_int8(fe, spec.dims, blob, spec.offset, alphas), orc.mlp(fe, spec.dims, blob, spec.offset)


def gpu_int8(B, cfg, batch, blob, alphas):
    etx = B.Etx(B.make_desc(cfg, precision=0), blob)
    db = B.DeviceBatch(batch, etx.device)
    emb = etx.etx_embed_int8(db, alphas)
    torch.cuda.synchronize()
    assert etx.launch_count() == 1
    return etx, db, emb


@pytest.mark.parametrize("name", ["c0", "c1"])
def test_int8_embedding_bit_equal_single_event(B, name):
    cfg = synth.CONFIGS[name]
    batch, blob = synth.generate_events(cfg), synth.generate_weights(cfg)
    alphas = synth.int8_act_alpha(cfg)
    want, e32 = oracle_int8(cfg, batch, blob, alphas)
    _, _, emb = gpu_int8(B, cfg, batch, blob, alphas)
    np.testing.assert_array_equal(emb.cpu().numpy().view(np.uint32), want.view(np.uint32))      # bit for bit
    assert 0 < np.abs(want - e32).max() < 0.15 * np.abs(e32).max()                               # a real quantisation, calibrated


def test_int8_embedding_batch_ragged_tail_clipping_and_graph(B):
    cfg = synth.CONFIGS["c2"]
    batch = synth.generate_events(cfg, range(200, 223))           # 23 events: several 64-row tiles and a ragged tail
    blob = synth.generate_weights(cfg)
    alphas = synth.int8_act_alpha(cfg)
    for al in (alphas, alphas * np.float32(0.25)):                # ranges 4x too narrow: the clip of Eq. 4.33 is exercised
        want, _ = oracle_int8(cfg, batch, blob, al)
        etx, db, emb = gpu_int8(B, cfg, batch, blob, al)
        np.testing.assert_array_equal(emb.cpu().numpy().view(np.uint32), want.view(np.uint32))
    # the graph built from the INT8 embedding equals the oracle's graph from the oracle's INT8 embedding
    r2, gap = synth.r2_max(cfg), cfg.max_plane_gap
    want, e32 = oracle_int8(cfg, batch, blob, alphas)
    s8, d8 = orc.build_graph(batch["event_ptr"], batch["plane"], want, r2, gap)
    s32, _ = orc.build_graph(batch["event_ptr"], batch["plane"], e32, r2, gap)
    etx, db, emb = gpu_int8(B, cfg, batch, blob, alphas)
    cap = len(s8) + 16
    etx.ensure_workspace(db.n_events, db.n_hits, cap)
    g = B.DeviceGraph(db.n_hits, cap, etx.device)
    E = etx.etx_build_graph(db, emb, r2, gap, g)
    assert E == len(s8)
    np.testing.assert_array_equal(g.src[:E].cpu().numpy(), s8)
    np.testing.assert_array_equal(g.dst[:E].cpu().numpy(), d8)
    print(f"INT8 embedding: {len(s8)} edges vs {len(s32)} from the fp32 embedding ({len(s8) / len(s32):.3f}x; thesis P:2742: 1.05-1.10x)")


def test_int8_embedding_other_width_and_errors(B):
    cfg = dataclasses.replace(synth.CONFIGS["c0"], emb_widths=(3, 64, 64, 3))        # H = 64, d = 3
    batch, blob = synth.generate_events(cfg), synth.generate_weights(cfg)
    spec = synth.model_layout(cfg)[0]
    fe, _ = orc.features(batch, synth.NORM_CENTER, synth.NORM_SCALE)
    alphas = orc.int8_calibration(fe, spec.dims, blob, spec.offset)
    want = orc.mlp_int8(fe, spec.dims, blob, spec.offset, alphas)
    etx, db, emb = gpu_int8(B, cfg, batch, blob, alphas)
    np.testing.assert_array_equal(emb.cpu().numpy().view(np.uint32), want.view(np.uint32))
    with pytest.raises(B.EtxError) as ei:
        etx.etx_embed_int8(db, alphas[:-1])                                          # one range per layer
    assert ei.value.status == B.ETX_ERR_INVALID
    with pytest.raises(B.EtxError) as ei:
        etx.etx_embed_int8(db, alphas * 0)                                           # ranges must be positive
    assert ei.value.status == B.ETX_ERR_INVALID
