"""B200-native device-resident decoder for ACEAPEX-style absolute-offset LZ77 archives (arxiv 2606.18900).

The product is the CUDA library behind include/aceapex.h; `paper_2606_18900_b200.aceapex` is its thin binding.
`datagen` (synthetic inputs) and `encoder` (archive writer) only produce test inputs."""
