"""bench.py's algorithmic byte / flop counts (-m "not gpu") against the per-config figures of SURVEY.md 8(d) -- the
roofline fractions of the bench line are these counts divided by measured times, so a slip here would silently
move every reported fraction."""
import gen
import bench


def test_update_bytes_match_the_survey_table():
    c3, c5, c2 = gen.spec_for("c3"), gen.spec_for("c5"), gen.spec_for("c2")
    # U = min(T, K_max) touched prototypes -> C3 146.6 MB, C5 212 MB, C2 5.2 MB per frame
    assert abs(bench.update_bytes_per_frame(c3, min(c3.T, c3.k_max)) / 1e6 - 146.6) < 0.5
    assert abs(bench.update_bytes_per_frame(c5, min(c5.T, c5.k_max)) / 1e6 - 212) < 1.5
    assert abs(bench.update_bytes_per_frame(c2, min(c2.T, c2.k_max)) / 1e6 - 5.2) < 0.05
    # per bank: 6 T d elt + K (4 d + 40) + U (16 d + 80) + 16 G T
    per_bank = 6 * 196 * 128 * 2 + 1024 * (4 * 128 + 40) + 196 * (16 * 128 + 80) + 16 * 8 * 196
    assert bench.update_bytes_per_frame(c2, 196) == per_bank * 4


def test_query_flops_and_assignment_flops():
    c3, c5 = gen.spec_for("c3"), gen.spec_for("c5")
    fact, dense = bench.query_flops(c3)
    # C3 60 / 146 GF (factorised / dense-equivalent), C5 64 / 176 GF; with the bank's K_max = 1024 the
    # factorised count is 4 rows (W + K_max) d
    assert abs(dense / 1e9 - 145.5) < 0.5 and abs(fact / 1e9 - 53.4) < 0.5
    rows, W, L = 224, 16 * 196, 16 * 196 + 1024 * 8
    assert dense == 4.0 * rows * L * 128 * 112 and fact == 4.0 * rows * (W + 1024) * 128 * 112
    fact5, dense5 = bench.query_flops(c5)
    assert abs(dense5 / 1e9 - 176.1) < 0.5
    # assignment: 2 T K_max d per bank-frame (x2 on the tensor pipe with the hi + lo split): C3 5.75 GF, C5 19.3 GF
    assert abs(bench.assign_flops_per_frame(c3) / 1e9 - 5.755) < 0.01
    assert abs(bench.assign_flops_per_frame(c5) / 1e9 - 19.33) < 0.01


def test_query_bytes_count_fp32_centres_and_codes():
    c3 = gen.spec_for("c3")
    per_bank = 2 * 3136 * 128 * 2 + 1024 * (2 * 128 * 4 + 8 * 8 + 4) + 2 * 224 * 128 * 2
    assert bench.query_bytes(c3) == per_bank * 112


def test_decode_bytes_count_the_centres_at_the_streamed_width():
    c3 = gen.spec_for("c3")
    per_bank = 2 * 3136 * 128 * 2 + 1024 * (2 * 128 * 2 + 8 * 8 + 4) + 2 * 7 * 128 * 2
    assert bench.decode_bytes(c3, 2) == per_bank * 112
    assert bench.decode_bytes(c3, 4) - bench.decode_bytes(c3, 2) == 1024 * 2 * 128 * 2 * 112


def test_peaks_fall_back_when_the_driver_file_is_absent(tmp_path, monkeypatch):
    monkeypatch.setattr(bench, "ROOT", str(tmp_path))
    p = bench.load_peaks()
    assert p["source"] == "fallback" and p["hbm"] > 6000 and p["bf16_sustained"] < p["bf16_burst"]
