import sys, torch
sys.path.insert(0, str(__import__('pathlib').Path(__file__).resolve().parents[2]))
from paper_2607_01237_b200 import kara
kara.lib()
dev = torch.device('cuda:0')
T, Dm, Hq, d = 32768, 5120, 40, 128
hid = torch.randn(T, Dm, device=dev).to(torch.bfloat16)
wq = (torch.randn(Hq * d, Dm, device=dev) / Dm ** 0.5).to(torch.bfloat16)
pos = (torch.arange(T, device=dev, dtype=torch.int32) % 512) + 20000
out = torch.empty(T, Hq, d, dtype=torch.bfloat16, device=dev)
for _ in range(4):
    kara.kara_window_queries(hid, wq, pos, 1e6, Hq, d, out=out, max_position=32768)
torch.cuda.synchronize()
print("ok")
