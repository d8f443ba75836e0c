"""Pin P14: bench.py's byte / FLOP formulas reproduce the totals the paper prints."""
import os

from paper_2606_26439_b200 import accounting as acc

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "paper_io_totals.txt")


def golden():
    out = {}
    for line in open(GOLDEN):
        line = line.split("#")[0].split()
        if len(line) == 2:
            out[line[0]] = float(line[1])
    return out


def test_dense_io_model_matches_printed_totals():
    g = golden()
    B, Nq, Nd, d = 10**4, 32, 128, 128
    assert acc.io_naive_eq4(B, Nq, Nd, d) == g["naive_io_bytes"]
    assert acc.io_fused_eq5(B, Nq, Nd, d) == g["fused_io_bytes"]
    fl = acc.flops_eq3(B, Nq, Nd, d)
    assert round(fl / acc.io_naive_eq4(B, Nq, Nd, d), 1) == g["naive_ai"]
    assert round(fl / acc.io_fused_eq5(B, Nq, Nd, d), 1) == g["fused_ai"]
    assert round(acc.io_naive_eq4(B, Nq, Nd, d) / acc.io_fused_eq5(B, Nq, Nd, d), 1) == g["io_reduction"]
    assert round(acc.io_naive_eq4(B, 64, Nd, d) / acc.io_fused_eq5(B, 64, Nd, d), 1) == g["io_reduction_nq64"]


def test_pq_io_model_matches_printed_totals():
    g = golden()
    B, Nq, Nd, d, M, K = 10**5, 32, 128, 128, 16, 256
    assert acc.pq_io_decompress_then_score(B, Nq, Nd, d, M) == g["pq_decompress_io_bytes"]
    assert acc.pq_io_fused(B, Nq, Nd, M, K) == g["pq_fused_io_bytes"]
    assert round(g["pq_decompress_io_bytes"] / g["pq_fused_io_bytes"], 1) == g["pq_io_ratio"]
    assert Nq * M * K * 4 == g["pq_table_bytes"]


def test_generalised_formulas_reduce_to_the_papers_at_q1_uniform():
    g = golden()
    B, Nq, Nd, d = 10**5, 32, 128, 128
    assert acc.dense_bytes(1, Nq, d, B * Nd, B, 2) == acc.io_optimal_eq7(B, Nq, Nd, d)
    assert acc.pq_bytes(1, Nq, 16, 256, B * Nd, B) == acc.pq_io_fused(B, Nq, Nd, 16, 256) - B * Nq * 4 + B * 4
    # Table 7 at B=100K, 1.232 ms: 2,660 GB/s and 85.1 TFLOP/s
    assert round(acc.dense_bytes(1, Nq, d, B * Nd, B, 2) / 1.232e-3 / 1e9) == g["table7_gbs_100k"]
    assert round(acc.dense_flops(1, Nq, d, B * Nd) / 1.232e-3 / 1e12, 1) == g["table7_tflops_100k"]
