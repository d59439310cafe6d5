"""Pin P1: the oracle against the values PRINTED in FIPS-197 and SP 800-38A.

Fixtures and their citations are in tests/golden/ (see its README.md).  These
pin the key schedule, each round transformation in isolation (Appendix C.1's
round trace), the whole cipher for the three key sizes, and CTR chaining with a
counter whose low byte carries (the F.5 counter ends in ...fe ff -> ff 00).
"""
import pytest

from oracle import oracle as o


def test_fips197_appendix_b_and_c_ciphertexts(golden):
    g = golden("fips197_appendix_c.txt")
    assert o.encrypt_block(g["b.key"], g["b.input"]) == g["b.output"]
    for tag in ("c1", "c2", "c3"):
        key, want = g[tag + ".key"], g[tag + ".output"]
        assert o.encrypt_block(key, g["c.plaintext"]) == want
        assert o.decrypt_block(key, want) == g["c.plaintext"]


def test_fips197_c1_round_trace_pins_each_transformation(golden):
    g = golden("fips197_appendix_c.txt")
    rk, nr = o.key_expand(g["c1.key"])
    assert nr == 10
    # round[0]: input xor k_sch = round[1].start
    assert o.add_round_key(g["c.plaintext"], rk[0:16]) == g["c1.round1.start"]
    assert o.sub_bytes(g["c1.round1.start"]) == g["c1.round1.s_box"]
    assert o.shift_rows(g["c1.round1.s_box"]) == g["c1.round1.s_row"]
    assert o.mix_columns(g["c1.round1.s_row"]) == g["c1.round1.m_col"]
    assert rk[16:32] == g["c1.round1.k_sch"]
    assert o.add_round_key(g["c1.round1.m_col"], rk[16:32]) == g["c1.round2.start"]
    assert rk[160:176] == g["c1.round10.k_sch"]
    # and the inverse transformations undo the printed values
    assert o.inv_sub_bytes(g["c1.round1.s_box"]) == g["c1.round1.start"]
    assert o.inv_shift_rows(g["c1.round1.s_row"]) == g["c1.round1.s_box"]
    assert o.inv_mix_columns(g["c1.round1.m_col"]) == g["c1.round1.s_row"]


def test_fips197_appendix_a_key_expansion(golden):
    g = golden("fips197_appendix_a.txt")
    rk, nr = o.key_expand(g["a1.key"])
    assert (nr, len(rk)) == (10, 176)
    assert rk[:16] == g["a1.key"]
    assert rk[16:32] == g["a1.w4_w7"] and rk[160:176] == g["a1.w40_w43"]
    rk, nr = o.key_expand(g["a2.key"])
    assert (nr, len(rk)) == (12, 208)
    assert rk[24:28] == g["a2.w6"] and rk[192:208] == g["a2.w48_w51"]
    rk, nr = o.key_expand(g["a3.key"])
    assert (nr, len(rk)) == (14, 240)
    assert rk[32:36] == g["a3.w8"] and rk[224:240] == g["a3.w56_w59"]


@pytest.mark.parametrize("tag", ["f51", "f53", "f55"])
def test_sp800_38a_f5_ctr_vectors(golden, tag):
    g = golden("sp800_38a_f5_ctr.txt")
    key, icb, pt, ct = g[tag + ".key"], g["f5.init_counter"], g["f5.plaintext"], g[tag + ".ciphertext"]
    assert o.ctr(key, icb, pt) == ct          # Encrypt
    assert o.ctr(key, icb, ct) == pt          # Decrypt (F.5.2/4/6)
    # every prefix, including partial blocks: the leading bytes of the keystream block are used
    for n in (0, 1, 15, 16, 17, 31, 33, 63):
        assert o.ctr(key, icb, pt[:n]) == ct[:n]
    # random access: block j alone, started at icb + j
    for j in range(4):
        assert o.ctr(key, icb, pt[16 * j:16 * j + 16], block_offset=j) == ct[16 * j:16 * j + 16]


def test_sp800_38a_f51_input_and_output_blocks(golden):
    g = golden("sp800_38a_f5_ctr.txt")
    icb = g["f5.init_counter"]
    assert o.ctr_add(icb, 0) == icb
    assert o.ctr_add(icb, 1) == g["f51.input_block2"]
    assert o.ctr_add(icb, 2) == g["f51.input_block3"]
    assert o.ctr_add(icb, 3) == g["f51.input_block4"]
    # keystream = CTR of zeros = the printed "Output Block"s
    assert o.ctr(g["f51.key"], icb, bytes(64)) == g["f51.output_blocks"]
    for j in range(4):
        blk = o.encrypt_block(g["f51.key"], o.ctr_add(icb, j))
        assert blk == g["f51.output_blocks"][16 * j:16 * j + 16]
