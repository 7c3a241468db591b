"""One call of the FP8 path at the C1 shape (8 experts x 1024 rows): quantise, pack, run.  Used as the
command of the ncu capture in profiles/r1_ffn_fp8_ncu.md;  python -m paper_2606_00735_b200.fp8_demo"""
import torch

from . import binding as B


def main(E=8, d=4096, f=14336, n=1024, iters=6):
    B.load()
    W1 = (torch.randn((E, d, f), device="cuda") * d ** -0.5).to(torch.bfloat16)
    W3 = (torch.randn((E, d, f), device="cuda") * d ** -0.5).to(torch.bfloat16)
    W2 = (torch.randn((E, f, d), device="cuda") * f ** -0.5).to(torch.bfloat16)
    W1q, s1 = B.fp8_pack_weights(W1)
    W3q, s3 = B.fp8_pack_weights(W3)
    W2q, s2 = B.fp8_pack_weights(W2)
    Xp = torch.randn((E * n, d), device="cuda").to(torch.bfloat16)
    off = (torch.arange(E + 1, device="cuda", dtype=torch.int32) * n).contiguous()
    hs = torch.full((E,), 8.0 / 448.0, dtype=torch.float32, device="cuda")
    for _ in range(iters):
        Xq, rs = B.fp8_quantize_rows(Xp)
        Y, Hq = B.grouped_ffn_fp8(Xq, rs, off, W1q, s1, W3q, s3, W2q, s2, hs)
    torch.cuda.synchronize()
    print("fp8 demo ok", float(Y.float().abs().mean()))


if __name__ == "__main__":
    main()
