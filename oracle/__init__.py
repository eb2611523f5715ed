"""CPU oracle for the MLP-Splatting forward render -- TEST INFRASTRUCTURE ONLY.

Importers allowed: tests/, __graft_entry__.smoke(), bench.py's cpu_baseline and
`--impl reference` legs.  Nothing under paper_2606_03877_b200/ may import this.
"""
