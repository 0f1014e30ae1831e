"""The flop counts behind bench.py's roofline fraction (flop_model.json) were captured under ncu on particular kernel
builds.  bench.py prints a fraction only when the loaded library's kernels are the captured ones; this test says so
without a GPU: every entry's fingerprint equals the fingerprint of the kernel sources and compiler flags in the tree
(paper_1501_03450_b200/build.py: kernel_source_hash), its capture file exists, and the model has the headline entry."""
import json
import os

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_flop_model_was_captured_on_the_kernel_sources_in_the_tree():
    from paper_1501_03450_b200 import build
    have = build.kernel_source_hash()
    model = json.load(open(os.path.join(ROOT, "flop_model.json")))
    assert "cfg3_rhic_like_bend_kick_n8_d4" in model
    for key, entry in model.items():
        cap = entry["capture"]
        assert cap["kernel_info"]["source_hash"] == have, (key, cap["kernel_info"]["source_hash"], have)
        assert os.path.exists(os.path.join(ROOT, entry["source"])), entry["source"]
        fp64 = entry["dfma_per_particle_turn"] + entry["dadd_per_particle_turn"] + entry["dmul_per_particle_turn"]
        assert abs(fp64 - entry["fp64_inst_per_particle_turn"]) < 1e-6 * fp64
        flop = 2 * entry["dfma_per_particle_turn"] + entry["dadd_per_particle_turn"] + entry["dmul_per_particle_turn"]
        assert abs(flop - entry["flop_per_particle_turn"]) < 1e-6 * flop
