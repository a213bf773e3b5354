"""Writes the closed-form fixtures of tests/golden/.  Uses only Python's math module — neither oracle/
nor the CUDA path — so the stored values are independent of both."""
import math
import os

HERE = os.path.dirname(os.path.abspath(__file__))


def main():
    # attention, Nq = 2, Nk = 2, H = 1, d = 1, scale = 1: p_i0 = 1 / (1 + exp(q_i (k1 - k0)))
    q, k, v = [0.5, -2.0], [1.0, -1.0], [3.0, 7.0]
    with open(os.path.join(HERE, "attention_2x2_closed_form.txt"), "w") as f:
        f.write("# q0 q1 | k0 k1 | v0 v1 | o0 o1 | lse0 lse1 ; o_i = p v0 + (1-p) v1, p = 1/(1+exp(q_i (k1-k0))), "
                "lse_i = log(exp(q_i k0) + exp(q_i k1)); scale = 1 (SURVEY 8(c) step 5)\n")
        o, lse = [], []
        for qi in q:
            p = 1.0 / (1.0 + math.exp(qi * (k[1] - k[0])))
            o.append(p * v[0] + (1 - p) * v[1])
            lse.append(math.log(math.exp(qi * k[0]) + math.exp(qi * k[1])))
        f.write(" ".join(repr(x) for x in q + k + v + o + lse) + "\n")
    with open(os.path.join(HERE, "gelu_tanh_points.txt"), "w") as f:
        f.write("# z gelu_tanh(z) = 0.5 z (1 + tanh(0.7978845608028654 (z + 0.044715 z^3)))  (SURVEY 8(c) step 5)\n")
        for z in (-3.0, -1.0, -0.25, 0.0, 0.5, 1.0, 2.0, 6.0):
            f.write(f"{z!r} {0.5 * z * (1 + math.tanh(0.7978845608028654 * (z + 0.044715 * z ** 3)))!r}\n")
    with open(os.path.join(HERE, "rope_points.txt"), "w") as f:
        f.write("# j cos(3 w_j) sin(3 w_j), w_j = 10000^(-2j/8): image of the pair (1,0) at pos 3, d_a = 8 (R6)\n")
        for j in range(4):
            w = 10000.0 ** (-2.0 * j / 8)
            f.write(f"{j} {math.cos(3 * w)!r} {math.sin(3 * w)!r}\n")


if __name__ == "__main__":
    main()
